"""`-m gpu` parity tests of the vision-tower front end (te_encode_image, te_config.non_causal)
against oracle/te_vision.py on the same seeded pixels and weights.  Everything goes through the C ABI.

Gates.  Each stage feeds bf16-rounded operands to an fp32-accumulating GEMM, like the decoder: the patch embedding
rounds the pixels (|err| <= 2^-9 relative per element -> rel-L2 ~ 2e-3 of x0), the tower is the decoder's block (update
floor 3.7e-3 per layer), the merger rounds the normalised tower output.  Whole-tensor rel-L2 <= 1e-2 per
stage and max per-row rel-L2 <= 2.5e-2 (tests/parity_metrics.py: the same per-layer / per-row bounds as the decoder's).
"""
import numpy as np
import pytest

import workloads as W
import parity_metrics as PM

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def O():
    from oracle import te_oracle
    return te_oracle


@pytest.fixture(scope="module")
def V():
    from oracle import te_vision
    return te_vision


@pytest.fixture(scope="module")
def H():
    import gpu_helpers
    return gpu_helpers


def _split(v, blob):
    lay = W.vision_blob_layout(v)
    w_pe = blob[lay["W_pe"][0]:lay["W_pe"][0] + int(np.prod(lay["W_pe"][1]))].reshape(lay["W_pe"][1])
    tower = blob[lay["tower"][0]:lay["tower"][0] + lay["tower"][1]]
    w_m = blob[lay["W_m"][0]:lay["W_m"][0] + int(np.prod(lay["W_m"][1]))].reshape(lay["W_m"][1])
    return w_pe, tower, w_m


def _run_gpu(v, blob, px, text_lens=None, d_text_fill=None):
    """te_encode_image through the binding; returns (embeds, taps, launches)."""
    import torch
    import paper_2606_05981_b200 as te
    B = px.shape[0]
    n_vis = v.tokens_per_frame
    enc = te.VisionEncoder(v, B)
    enc.load_weights(blob)
    pd = torch.from_numpy(np.ascontiguousarray(px, dtype=np.float32)).cuda()
    tl = None if text_lens is None else torch.from_numpy(np.asarray(text_lens, dtype=np.int32)).cuda()
    T = B * n_vis + (0 if text_lens is None else int(np.sum(text_lens)))
    emb = torch.full((T, v.out_hidden), -7.0 if d_text_fill is None else d_text_fill, dtype=torch.float32, device="cuda")
    enc.encode_image(B, pd, tl, emb)
    torch.cuda.synchronize()
    n_patch = B * v.grid_h * v.grid_w
    taps = {}
    for name, what, shape in (("patch_embeds", te.TE_VTAP_PATCH_EMBEDS, (n_patch, v.tower.hidden)),
                              ("tower_out", te.TE_VTAP_TOWER_OUT, (n_patch, v.tower.hidden)),
                              ("merged", te.TE_VTAP_MERGED, (B * n_vis, v.out_hidden))):
        buf = np.empty(shape, dtype=np.float32)
        te.te_vision_debug_tap(enc.v, what, buf)
        taps[name] = buf
    launches = te.te_vision_kernel_launches(enc.v)
    tower = te.te_vision_debug_tower(enc.v)
    assert te.te_query_async_error(tower) == te.TE_OK
    # the tower's rotary ids (0, py, px) bit-exact and its cos/sin table (what an h / w swap would show in; the outputs
    # barely move under it, tests/test_vision_pins.py)
    from oracle import te_oracle as O_
    pos = np.empty((3, n_patch), dtype=np.int32)
    te.te_debug_tap(tower, te.TE_TAP_POS, pos)
    want = O_.position_ids([0] * B, v.grid_h, v.grid_w)
    assert np.array_equal(pos, want)
    hd2 = v.tower.head_dim // 2
    cos_t = np.empty((n_patch, hd2), dtype=np.float32)
    te.te_debug_tap(tower, te.TE_TAP_COS, cos_t)
    phi = O_.mrope_angles(want, v.tower.head_dim, v.tower.rope_sections, v.tower.rope_theta)
    assert np.max(np.abs(cos_t - np.cos(phi))) <= PM.GATE_COSSIN_ABS
    out = emb.cpu().numpy()
    enc.close()
    return out, taps, launches


def _check_stages(v, V, blob, px, taps, tag):
    w_pe, tower, w_m = _split(v, blob)
    ot = {}
    ref = V.encode_image(w_pe, tower, W.blob_layout(v.tower), v.tower, w_m, px, v.patch, taps=ot)
    for name, want in (("patch_embeds", ot["patch_embeds"]), ("tower_out", ot["tower_out"]), ("merged", ref)):
        got = taps[name].astype(np.float64)
        assert np.isfinite(got).all(), (tag, name)
        assert PM.rel_l2(got, want) <= PM.GATE_LAYER_REL_L2, (tag, name, PM.rel_l2(got, want))
        assert PM.max_row_rel_l2(got, want) <= PM.GATE_ROW_UPDATE_REL_L2, (tag, name, PM.max_row_rel_l2(got, want))
    return ref


def test_vision_tiny_all_stages(V):
    """CPU-sized front end (32x32 image, 8x8 patches, d_v = 128, 2 tower layers, merger to 256): every stage."""
    v = W.VISION_TINY
    blob = W.make_vision_blob(v)
    px = W.make_pixels(v, 2)
    out, taps, launches = _run_gpu(v, blob, px)
    ref = _check_stages(v, V, blob, px, taps, "tiny")
    assert np.array_equal(out, taps["merged"])                       # no text: embeds = the merged tokens, packed
    assert PM.rel_l2(out, ref) <= PM.GATE_LAYER_REL_L2
    # patchify + GEMM + (refresh + prep + 5 per layer + final norm) + merge + GEMM + scatter
    assert launches == 5 + (2 + 5 * v.tower.n_layers + 1)


def test_vision_scatter_into_packed_embeds(V):
    """With the decoder's text_lens the merged tokens land on rows cu[b] .. cu[b] + n_vis; text rows are untouched."""
    v = W.VISION_TINY
    blob = W.make_vision_blob(v)
    B = 3
    px = W.make_pixels(v, B)
    tl = np.asarray([5, 0, 9], dtype=np.int32)
    out, taps, _ = _run_gpu(v, blob, px, text_lens=tl, d_text_fill=123.0)
    n_vis = v.tokens_per_frame
    row = 0
    for b in range(B):
        assert np.array_equal(out[row:row + n_vis], taps["merged"][b * n_vis:(b + 1) * n_vis]), b
        assert np.all(out[row + n_vis:row + n_vis + tl[b]] == 123.0), b
        row += n_vis + tl[b]
    assert row == out.shape[0]


@pytest.mark.parametrize("B", [1, 5])
def test_vision_full_shape(V, B):
    """The paper's shape: 256x256 source patch -> 16x16 patches of 16x16 pixels -> 8x8 = 64 visual tokens of width 2048
    (PAPER.md:23); tower d_v = 1024, 16 heads of 64, 4 layers.  B = 5: 1280 patch rows = CTA-pair tiles with a ragged
    last row block; B = 1: one-CTA tiles and the split-K kernels inside the tower."""
    v = W.VISION_FULL
    blob = W.make_vision_blob(v)
    px = W.make_pixels(v, B)
    out, taps, _ = _run_gpu(v, blob, px)
    ref = _check_stages(v, V, blob, px, taps, f"full B={B}")
    assert out.shape == (B * 64, 2048)
    assert PM.rel_l2(out, ref) <= PM.GATE_LAYER_REL_L2
    assert PM.cos_sim(out, ref) > 0.9999


def test_vision_bench_shape_all_frames(V):
    """B = 16 (cfg 4's frames): 4096 patch rows through the CTA-pair / wide-tile dispatch; every frame compared."""
    v = W.VISION_FULL
    blob = W.make_vision_blob(v)
    px = W.make_pixels(v, 16)
    out, taps, _ = _run_gpu(v, blob, px)
    ref = _check_stages(v, V, blob, px, taps, "full B=16")
    assert PM.max_row_rel_l2(out, ref) <= PM.GATE_ROW_UPDATE_REL_L2


def test_vision_frames_independent_and_order_visible():
    """A frame's visual tokens do not depend on its batch neighbours (bitwise: same tiles, same order of operations
    inside a frame's rows is NOT guaranteed across batch sizes, so compare within tolerance 1e-5), and swapping two pixel
    patches inside one merged cell moves that frame's tokens (the merge order is live on the device)."""
    v = W.VISION_TINY
    blob = W.make_vision_blob(v)
    px = W.make_pixels(v, 3)
    out, _, _ = _run_gpu(v, blob, px)
    n_vis = v.tokens_per_frame
    solo, _, _ = _run_gpu(v, blob, px[1:2])
    assert np.max(np.abs(out[n_vis:2 * n_vis] - solo)) <= 1e-5 * np.max(np.abs(solo))
    px2 = px.copy()
    P = v.patch
    px2[0, :P, :P], px2[0, :P, P:2 * P] = px[0, :P, P:2 * P].copy(), px[0, :P, :P].copy()
    out2, _, _ = _run_gpu(v, blob, px2)
    assert not np.allclose(out2[:n_vis], out[:n_vis], rtol=1e-3, atol=1e-4)
    assert np.array_equal(out2[n_vis:], out[n_vis:])


@pytest.mark.parametrize("attn_impl", [1, 0])
@pytest.mark.parametrize("text_lens", [[24, 24], [0, 37, 5]])
def test_non_causal_decoder_stack(O, V, H, attn_impl, text_lens):
    """te_config.non_causal on the decoder-shaped tiny stack WITH text tokens and ragged frames, on both attention
    kernels (tcgen05 / mma.sync): the oracle is te_oracle.encode with te_vision.attention_full_gqa.  The causal result
    must be far away (the flag is live)."""
    w = W.get_workload(1)
    m = w.model
    blob = H.cached_blob(m, w.seed_weights)
    tl = np.asarray(text_lens, dtype=np.int32)
    T = int(np.sum(tl)) + len(tl) * w.grid_h * w.grid_w
    emb = W.make_embeddings(w, T)
    g = H.GpuTE(m, len(tl), T, blob, attn_impl=attn_impl, non_causal=1)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    g.close()
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, attention=V.attention_full_gqa)
    mm = PM.stack_metrics(out, ref, emb)
    assert PM.passes_final_gates(mm), mm
    causal = O.encode(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w)
    assert PM.rel_l2(out - emb, causal - emb) > 10 * mm["update_rel_l2"]


def test_image_to_hidden_states_end_to_end(O, V, H):
    """TE(x, p) -> h with the frame itself as input: te_encode_image writes the visual rows of the
    decoder's packed input on the device, te_encode consumes them; the oracle chains te_vision.encode_image and
    te_oracle.encode.  Tiny shapes: 4 visual tokens on a 2x2 grid + text."""
    import torch
    import paper_2606_05981_b200 as te
    v = W.VISION_TINY
    w = W.get_workload(1)
    m = w.model
    assert v.out_hidden == m.hidden
    vblob = W.make_vision_blob(v)
    blob = H.cached_blob(m, w.seed_weights)
    B = 2
    tl = np.asarray([24, 11], dtype=np.int32)
    gh, gw = v.grid_h // 2, v.grid_w // 2
    n_vis = gh * gw
    T = B * n_vis + int(tl.sum())
    px = W.make_pixels(v, B)
    emb = W.make_embeddings(w, T)                    # the text rows are taken from here
    venc = te.VisionEncoder(v, B)
    venc.load_weights(vblob)
    dec = te.TextEncoder(m, B, T)
    dec.load_weights(blob)
    e = torch.from_numpy(emb).cuda()
    lens = torch.from_numpy(tl).cuda()
    out = torch.empty_like(e)
    venc.encode_image(B, torch.from_numpy(px).cuda(), lens, e)       # same stream, no sync in between
    dec.encode(B, gh, gw, e, lens, T, out)
    torch.cuda.synchronize()
    assert te.te_query_async_error(dec.h) == te.TE_OK
    got = out.cpu().numpy()
    got_emb = e.cpu().numpy()
    venc.close()
    dec.close()
    w_pe, tower, w_m = _split(v, vblob)
    vis = V.encode_image(w_pe, tower, W.blob_layout(v.tower), v.tower, w_m, px, v.patch)
    ref_emb = emb.astype(np.float64).copy()
    row = 0
    for b in range(B):
        ref_emb[row:row + n_vis] = vis[b * n_vis:(b + 1) * n_vis]
        row += n_vis + tl[b]
    assert PM.rel_l2(got_emb, ref_emb) <= PM.GATE_LAYER_REL_L2
    ref = O.encode(blob, W.blob_layout(m), m, ref_emb, tl, gh, gw)
    mm = PM.stack_metrics(got, ref, ref_emb)
    assert mm["rel_l2"] <= PM.GATE_FINAL_REL_L2 and mm["update_rel_l2"] <= PM.GATE_UPDATE_REL_L2, mm
    assert mm["max_row_update_rel_l2"] <= PM.GATE_ROW_UPDATE_REL_L2, mm


def test_encode_image_never_writes_past_total_tokens():
    """te_encode_image reads text_lens on the device, unvalidated: whatever it holds, no row at or past total_tokens may
    be written (te.h containment promise, same as te_encode), and the sticky flag must say what was wrong.  A guard band
    behind `embeds` shows any stray write."""
    import torch
    import paper_2606_05981_b200 as te
    v = W.VISION_TINY
    B, n_vis, d, guard = 3, v.tokens_per_frame, v.out_hidden, 64
    good = [5, 0, 7]
    T = B * n_vis + sum(good)
    enc = te.VisionEncoder(v, B)
    enc.load_weights(W.make_vision_blob(v))
    pd = torch.from_numpy(np.ascontiguousarray(W.make_pixels(v, B), dtype=np.float32)).cuda()

    def run(lens):
        buf = torch.full((T + guard, d), -7.0, dtype=torch.float32, device="cuda")
        tl = torch.tensor(lens, dtype=torch.int32, device="cuda")
        enc.encode_image(B, pd, tl, buf, total_tokens=T)
        rc = enc.query_async_error()
        return buf.cpu().numpy(), rc, te.lib().te_vision_last_error(enc.v).decode()

    ref, rc, _ = run(good)
    assert rc == te.TE_OK
    cu = np.concatenate([[0], np.cumsum([n_vis + t for t in good])])
    vis_rows = np.concatenate([np.arange(cu[b], cu[b] + n_vis) for b in range(B)])
    text_rows = np.setdiff1d(np.arange(T + guard), vis_rows)
    assert np.all(ref[text_rows] == -7.0) and not np.any(ref[vis_rows] == -7.0)

    # frame 1 claims 1000 text tokens: frame 2's visual rows would land ~1000 rows past the buffer
    got, rc, msg = run([5, 1000, 7])
    assert rc == te.TE_ERR_DEVICE_CHECK and "0x2" in msg, msg
    assert np.all(got[T:] == -7.0)                                         # guard band intact
    assert np.array_equal(got[:cu[2]], ref[:cu[2]])                        # frames 0 and 1 as before
    assert np.all(got[cu[2]:T] == -7.0)                                    # frame 2: skipped, not misplaced
    # partly out of range: frame 2 starts 10 rows late, so its last 3 visual rows fall off the end (7 text rows absorb the rest)
    got, rc, msg = run([5, 10, 7])
    assert rc == te.TE_ERR_DEVICE_CHECK and "0x2" in msg, msg
    assert np.all(got[T:] == -7.0)
    assert np.array_equal(got[cu[2] + 10:T], ref[cu[2]:cu[2] + n_vis][:T - cu[2] - 10])
    # negative length: counted as 0 and flagged as such (9 + 0 + 3 still adds up to the 12 text rows: bit 1 alone)
    got, rc, msg = run([9, -4, 3])
    assert rc == te.TE_ERR_DEVICE_CHECK and "0x1 " in msg, msg
    assert np.all(got[T:] == -7.0)
    # the flag is cleared by the query: a good call afterwards is clean and identical to the first one
    again, rc, _ = run(good)
    assert rc == te.TE_OK and np.array_equal(again, ref)
    enc.close()


def test_vision_boundary_errors():
    import ctypes
    import paper_2606_05981_b200 as te
    L = te.lib()
    v = W.VISION_TINY
    cfg = te.make_vision_config(v, 2)
    bad = te.make_vision_config(v, 2)
    bad.image_h = 24                                    # not a multiple of 2 * patch
    assert te.te_vision_blob_bytes(bad) == 0
    h = ctypes.c_void_p()
    assert L.te_vision_create(ctypes.byref(bad), 0, ctypes.byref(h)) == te.TE_ERR_INVALID_ARG
    big = te.make_vision_config(W.VISION_FULL, 2)
    big.image_h = 512                                   # 32 x 16 patches > 256 per frame
    assert L.te_vision_create(ctypes.byref(big), 0, ctypes.byref(h)) == te.TE_ERR_UNSUPPORTED
    vh = te.te_vision_create(cfg)
    blob = W.make_vision_blob(v)
    assert L.te_encode_image(vh, 1, 1, 0, 1, 64, 0) == te.TE_ERR_NOT_LOADED
    assert L.te_vision_load_weights(vh, blob.ctypes.data, blob.nbytes - 2) == te.TE_ERR_BLOB_SIZE
    te.te_vision_load_weights(vh, blob)
    assert L.te_encode_image(vh, 3, 1, 0, 1, 4096, 0) == te.TE_ERR_INVALID_ARG      # n_frames > max_frames
    assert L.te_encode_image(vh, 1, 0, 0, 1, 4096, 0) == te.TE_ERR_INVALID_ARG      # null pixels
    assert L.te_encode_image(vh, 1, 1, 0, 1, 0, 0) == te.TE_ERR_INVALID_ARG         # total_tokens < n_frames * n_vis
    te.te_vision_destroy(vh)
    # non_causal and a cached prefix exclude each other
    c = te.make_config(W.get_workload(1).model, 2, 80, max_prefix_tokens=8, non_causal=1)
    assert L.te_create(ctypes.byref(c), 0, ctypes.byref(h)) == te.TE_ERR_INVALID_ARG


# ------------------------------------------------------------------ te_encode_ex: per-frame grids, bf16 embeddings
def test_per_frame_grids(O, H):
    """One (grid_h, grid_w) per frame on the device: frames are independent, so the
    oracle is te_oracle.encode frame by frame with that frame's grid.  ids bit-exact, stack within the gates; the
    frames' text ids start at max(gh, gw) of THEIR grid; a frame with an empty grid (text only) is allowed."""
    import torch
    import paper_2606_05981_b200 as te
    w = W.get_workload(1)
    m = w.model
    blob = H.cached_blob(m, w.seed_weights)
    grids = np.asarray([[4, 4], [2, 7], [8, 1], [0, 0], [3, 5]], dtype=np.int32)
    tl = np.asarray([24, 3, 0, 40, 17], dtype=np.int32)
    S = grids[:, 0] * grids[:, 1] + tl
    T = int(S.sum())
    emb = W.make_embeddings(w, T)
    enc = te.TextEncoder(m, len(tl), T)
    enc.load_weights(blob)
    e = torch.from_numpy(emb).cuda()
    out = torch.empty_like(e)
    enc.encode_ex(len(tl), torch.from_numpy(grids).cuda(), 0, 0, e, 0, torch.from_numpy(tl).cuda(), T, out)
    torch.cuda.synchronize()
    assert te.te_query_async_error(enc.h) == te.TE_OK
    pos = np.empty((3, T), dtype=np.int32)
    te.te_debug_tap(enc.h, te.TE_TAP_POS, pos)
    cu = np.empty(len(tl) + 1, dtype=np.int32)
    te.te_debug_tap(enc.h, te.TE_TAP_CU_SEQLENS, cu)
    got = out.cpu().numpy()
    lay = W.blob_layout(m)
    ref = np.empty((T, m.hidden))
    want_pos = np.empty((3, T), dtype=np.int64)
    r = 0
    for b in range(len(tl)):
        gh, gw = int(grids[b, 0]), int(grids[b, 1])
        rows = slice(r, r + int(S[b]))
        if gh * gw == 0:        # text-only frame: ids 0, 1, 2, ... (max(gh, gw) = 0); the oracle takes a 1x0 grid
            want_pos[:, rows] = np.arange(int(S[b]))[None, :]
            ref[rows] = _text_only(O, blob, lay, m, emb[rows])
        else:
            want_pos[:, rows] = O.position_ids([int(tl[b])], gh, gw)
            ref[rows] = O.encode(blob, lay, m, emb[rows], [int(tl[b])], gh, gw)
        r += int(S[b])
    assert np.array_equal(cu, np.concatenate([[0], np.cumsum(S)]))
    assert np.array_equal(pos, want_pos)
    mm = PM.stack_metrics(got, ref, emb)
    assert PM.passes_final_gates(mm), mm
    # an entry that makes a frame too long raises the device flag
    bad = grids.copy()
    bad[1] = [20, 20]
    L = te.lib()
    assert L.te_encode_ex(enc.h, len(tl), torch.from_numpy(bad).cuda().data_ptr(), 0, 0, e.data_ptr(), 0,
                          torch.from_numpy(tl).cuda().data_ptr(), T, out.data_ptr(), 0) == te.TE_OK
    assert te.te_query_async_error(enc.h) == te.TE_ERR_DEVICE_CHECK
    enc.close()


def _text_only(O, blob, lay, m, emb_rows):
    """A frame without visual tokens = a text sequence with ids t = h = w = 0, 1, 2, ... — what te_oracle.encode computes
    for a 0-token grid whose text starts at max(gh, gw) = 0; te_oracle takes it as grid 0 x 0."""
    return O.encode(blob, lay, m, emb_rows, [emb_rows.shape[0]], 0, 0)


def test_bf16_embeddings_equal_fp32_call(H):
    """embeds_dtype = 1: the bf16 embeddings are widened exactly, so the stack's output is BITWISE that of te_encode on
    the same (bf16-representable) fp32 values — one full-width layer, with the x1000 outlier channels of cfg 3's recipe."""
    import torch
    import paper_2606_05981_b200 as te
    w, blob, tl, T, emb, ch = H.workload_inputs(2, outliers="x1000")
    m = w.model
    bits = W.f32_to_bf16_bits(emb)
    emb_r = (bits.astype(np.uint32) << np.uint32(16)).view(np.float32).reshape(emb.shape)
    enc = te.TextEncoder(m, w.n_frames, T)
    enc.load_weights(blob)
    lens = torch.from_numpy(tl).cuda()
    e32 = torch.from_numpy(emb_r).cuda()
    e16 = torch.from_numpy(bits.view(np.int16).reshape(emb.shape)).cuda()
    o32, o16 = torch.empty_like(e32), torch.empty_like(e32)
    enc.encode(w.n_frames, w.grid_h, w.grid_w, e32, lens, T, o32)
    enc.encode_ex(w.n_frames, None, w.grid_h, w.grid_w, e16, 1, lens, T, o16)
    torch.cuda.synchronize()
    assert te.te_query_async_error(enc.h) == te.TE_OK
    assert torch.equal(o32, o16)
    assert te.te_graph_captures(enc.h) == 1          # same shape class: the second call replays the first graph
    enc.close()


def test_vision_handle_reuse_across_batch_sizes():
    """One front-end handle, calls with shrinking and growing frame counts (operand rows left by a larger call stay in
    the library's buffers; the tower replays one graph per shape class): every call equals a fresh handle's, bitwise."""
    import torch
    import paper_2606_05981_b200 as te
    v = W.VISION_TINY
    blob = W.make_vision_blob(v)
    px = W.make_pixels(v, 5)
    n_vis = v.tokens_per_frame
    enc = te.VisionEncoder(v, 5)
    enc.load_weights(blob)
    got = {}
    for B in (5, 2, 5, 1):
        pd = torch.from_numpy(px[:B]).cuda()
        emb = torch.zeros((B * n_vis, v.out_hidden), dtype=torch.float32, device="cuda")
        enc.encode_image(B, pd, None, emb)
        torch.cuda.synchronize()
        got.setdefault(B, []).append(emb.cpu().numpy())
    assert te.te_graph_captures(te.te_vision_debug_tower(enc.v)) <= 3
    enc.close()
    assert np.array_equal(got[5][0], got[5][1])
    for B in (2, 1):
        fresh, _, _ = _run_gpu(v, blob, px[:B])
        assert np.array_equal(got[B][0], fresh), B


def test_per_frame_grids_full_width_ragged(O, H):
    """te_encode_ex at full width in the large-batch dispatch (CTA pairs, wide residual tiles, tcgen05 attention sized for
    the longest frame the capacities allow): 32 frames with five different grids (square, wide, tall, odd, none) and
    ragged text, one layer, every row against the per-frame oracle; ids and offsets bit-exact."""
    import torch
    import paper_2606_05981_b200 as te
    m = W.FULL1
    blob = H.cached_blob(m, 1)
    rng = np.random.default_rng(77)
    shapes = np.asarray([[8, 8], [4, 16], [12, 5], [7, 9], [0, 0]], dtype=np.int32)
    grids = shapes[rng.integers(0, len(shapes), size=32)]
    tl = rng.integers(16, 97, size=32).astype(np.int32)
    S = grids[:, 0] * grids[:, 1] + tl
    T = int(S.sum())
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    emb[:, [5, 1500]] *= np.float32(1000.0)
    enc = te.TextEncoder(m, 32, T)
    enc.load_weights(blob)
    e = torch.from_numpy(emb).cuda()
    out = torch.empty_like(e)
    enc.encode_ex(32, torch.from_numpy(np.ascontiguousarray(grids)).cuda(), 0, 0, e, 0, torch.from_numpy(tl).cuda(), T, out)
    torch.cuda.synchronize()
    assert te.te_query_async_error(enc.h) == te.TE_OK
    pos = np.empty((3, T), dtype=np.int32)
    te.te_debug_tap(enc.h, te.TE_TAP_POS, pos)
    got = out.cpu().numpy()
    enc.close()
    lay = W.blob_layout(m)
    ref = np.empty((T, m.hidden))
    want_pos = np.empty((3, T), dtype=np.int64)
    r = 0
    for b in range(32):
        rows = slice(r, r + int(S[b]))
        gh, gw = int(grids[b, 0]), int(grids[b, 1])
        want_pos[:, rows] = O.position_ids([int(tl[b])], gh, gw)
        ref[rows] = O.encode(blob, lay, m, emb[rows], [int(tl[b])], gh, gw)
        r += int(S[b])
    assert np.array_equal(pos, want_pos)
    mm = PM.stack_metrics(got, ref, emb, outlier_ch=[5, 1500])
    assert PM.passes_final_gates(mm), mm


def test_vision_non_square_image(V):
    """A 32 x 64 image (4 x 8 patches -> 2 x 4 visual tokens): row-major patch order, (dy, dx) merge order and the (0, py, px)
    ids on a non-square grid (a transposed layout anywhere would pass on the square configs)."""
    import dataclasses
    v = dataclasses.replace(W.VISION_TINY, image_h=32, image_w=64)
    blob = W.make_vision_blob(v)
    px = W.make_pixels(v, 3)
    out, taps, _ = _run_gpu(v, blob, px)
    ref = _check_stages(v, V, blob, px, taps, "non-square")
    assert out.shape == (3 * 8, v.out_hidden)
    assert PM.rel_l2(out, ref) <= PM.GATE_LAYER_REL_L2
    v2 = dataclasses.replace(W.VISION_TINY, image_h=64, image_w=16)
    px2 = W.make_pixels(v2, 2)
    out2, taps2, _ = _run_gpu(v2, W.make_vision_blob(v2), px2)
    _check_stages(v2, V, W.make_vision_blob(v2), px2, taps2, "tall")
