"""`-m gpu` parity tests: the CUDA path, called through the C-ABI binding, against the fp64 oracle
on the same seeded inputs.  Gates: tests/parity_metrics.py (BASELINE.json:north_star + SURVEY §8c).
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
def H():
    import gpu_helpers
    return gpu_helpers


def _assert_final(m, tag=""):
    assert m["rel_l2"] <= PM.GATE_FINAL_REL_L2, (tag, m)
    assert m["update_rel_l2"] <= PM.GATE_UPDATE_REL_L2, (tag, m)
    assert m["nonoutlier_rel_l2"] <= PM.GATE_NONOUTLIER_REL_L2, (tag, m)
    assert m["outlier_maxabs_rel"] <= PM.GATE_OUTLIER_MAXABS, (tag, m)
    assert m["max_row_update_rel_l2"] <= PM.GATE_ROW_UPDATE_REL_L2, (tag, m)          # every token row
    assert m["maxabs_update_over_rms"] <= PM.GATE_MAXABS_UPDATE_OVER_RMS, (tag, m)    # every element
    assert m["cos_sim"] > 0.999, (tag, m)


# --------------------------------------------------------------------------- GEMM main loop
@pytest.mark.parametrize("pair", [0, 1])
@pytest.mark.parametrize("M,N,K,bn", [(128, 256, 64, 256), (1, 128, 64, 128), (300, 512, 256, 256),
                                       (300, 512, 256, 128), (517, 768, 832, 256), (3072, 2048, 2048, 256),
                                       (3072, 2048, 6144, 128), (3072, 2048, 6144, 256), (3072, 4096, 2048, 256),
                                       (512, 12288, 2048, 256), (1024, 2048, 2048, 256)])
def test_gemm_mainloop_vs_fp64_matmul(H, M, N, K, bn, pair):
    """TMA + tcgen05 main loop alone: several tiles, ragged M tail, K spanning >1 pipeline ring.
    pair: 0 = one CTA per tile, 1 = CTA pairs (cta_group::2, 256-row tiles)."""
    import torch
    import paper_2606_05981_b200 as te
    rng = np.random.default_rng(M * 7 + N)
    a = W.f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    b = W.f32_to_bf16_bits(rng.standard_normal((N, K)).astype(np.float32))
    ref = H.bf16_bits_to_f64(a).reshape(M, K) @ H.bf16_bits_to_f64(b).reshape(N, K).T
    ad = torch.from_numpy(a.view(np.int16)).cuda()
    bd = torch.from_numpy(b.view(np.int16)).cuda()
    c = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    te.te_debug_gemm(0, ad, bd, c, M, N, K, bn, pair)
    out = c.cpu().numpy()
    assert np.isfinite(out).all()
    # fp32 accumulation of exact bf16 products: error ~ sqrt(K) * 2^-24 relative to |a||b|
    assert PM.rel_l2(out, ref) < 1e-5
    assert np.max(np.abs(out - ref)) < 1e-4 * np.sqrt(K) * 4


@pytest.mark.parametrize("M,N,K,bn,splits", [(128, 256, 128, 256, 2), (1, 128, 128, 128, 2), (80, 512, 256, 128, 2),
                                              (300, 512, 832, 128, 4), (128, 768, 832, 256, 3),
                                              (128, 2048, 2048, 128, 8), (128, 2048, 6144, 128, 8),
                                              (512, 2048, 6144, 128, 2), (128, 4096, 2048, 128, 4),
                                              (128, 12288, 2048, 256, 3), (512, 4096, 2048, 128, 1)])
def test_gemm_splitk_vs_fp64_matmul(H, M, N, K, bn, splits):
    """Split-K kernel: `splits` CTAs per tile (uneven K-slices included), partial tiles through the L2
    scratch, fixed-order sum -> same result as one fp64 matmul, and bitwise repeatable."""
    import torch
    import paper_2606_05981_b200 as te
    rng = np.random.default_rng(M * 11 + N + splits)
    a = W.f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    b = W.f32_to_bf16_bits(rng.standard_normal((N, K)).astype(np.float32))
    ref = H.bf16_bits_to_f64(a).reshape(M, K) @ H.bf16_bits_to_f64(b).reshape(N, K).T
    ad = torch.from_numpy(a.view(np.int16)).cuda()
    bd = torch.from_numpy(b.view(np.int16)).cuda()
    outs = []
    for _ in range(2):
        c = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
        te.te_debug_gemm_splitk(0, ad, bd, c, M, N, K, bn, splits)
        outs.append(c.cpu().numpy())
    assert np.isfinite(outs[0]).all()
    assert PM.rel_l2(outs[0], ref) < 1e-5
    assert np.max(np.abs(outs[0] - ref)) < 1e-4 * np.sqrt(K) * 4
    assert np.array_equal(outs[0], outs[1])


@pytest.mark.parametrize("M,N,K,n_tiles", [(3072, 2048, 2048, 6), (3072, 2048, 6144, 6), (3733, 2048, 2048, 4),
                                           (2048, 2048, 6144, 9), (1500, 2048, 2048, 7), (593, 256, 768, 5),
                                           (300, 256, 256, 3), (256, 2048, 2048, 16)])
def test_gemm_wide_vs_fp64_matmul(H, M, N, K, n_tiles):
    """One-wave wide-tile kernel alone (te_gemm_wide.cuh, plain epilogue), elementwise against an fp64 matmul: the
    widths the stack's dispatch picks at cfg 4 (6 x 352) and cfg 5 (4 x 512), a partly out-of-range last tile
    (7 x 320 > 2048), a wholly out-of-range one (5 x 64 > 256), a ragged last row-pair block, one MMA narrower than
    the other tile widths (16 x 128)."""
    import torch
    import paper_2606_05981_b200 as te
    rng = np.random.default_rng(M * 3 + N + n_tiles)
    a = W.f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    b = W.f32_to_bf16_bits(rng.standard_normal((N, K)).astype(np.float32))
    ref = H.bf16_bits_to_f64(a).reshape(M, K) @ H.bf16_bits_to_f64(b).reshape(N, K).T
    ad = torch.from_numpy(a.view(np.int16)).cuda()
    bd = torch.from_numpy(b.view(np.int16)).cuda()
    c = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    te.te_debug_gemm_wide(0, ad, bd, c, M, N, K, n_tiles)
    out = c.cpu().numpy()
    assert np.isfinite(out).all()
    assert PM.rel_l2(out, ref) < 1e-5
    assert np.max(np.abs(out - ref)) < 1e-4 * np.sqrt(K) * 4


# ------------------------------------------------------------------- ids / packing / rotary table
@pytest.mark.parametrize("gh,gw,tl", [(4, 4, [24, 24]), (8, 8, [64]), (4, 16, [3, 0, 17]), (16, 4, [0, 9]),
                                      (1, 5, [1, 2, 3, 4, 5, 6, 7])])
def test_position_ids_bit_exact(H, O, gh, gw, tl):
    m = W.TINY.with_layers(1)
    blob = H.cached_blob(m, 1)
    T = len(tl) * gh * gw + sum(tl)
    g = H.GpuTE(m, len(tl), T, blob)
    emb = np.random.default_rng(0).standard_normal((T, m.hidden)).astype(np.float32)
    g.encode(emb, tl, gh, gw)
    t = g.taps(T, len(tl))
    assert np.array_equal(t["pos"], O.position_ids(tl, gh, gw))
    assert np.array_equal(t["cu_seqlens"], O.cu_seqlens(tl, gh, gw))
    phi = O.mrope_angles(O.position_ids(tl, gh, gw), m.head_dim, m.rope_sections, m.rope_theta)
    assert np.max(np.abs(t["cos"] - np.cos(phi))) <= PM.GATE_COSSIN_ABS
    assert np.max(np.abs(t["sin"] - np.sin(phi))) <= PM.GATE_COSSIN_ABS
    import paper_2606_05981_b200 as te
    assert te.te_query_async_error(g.enc.h) == 0
    g.close()


# ------------------------------------------------------------ per-layer taps + teacher-forced layers
@pytest.mark.parametrize("cfg_id", [1, 2])
def test_layer_taps_and_teacher_forced_updates(H, O, cfg_id):
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    lay = W.blob_layout(m)
    g = H.GpuTE(m, w.n_frames, T, blob)
    x_in = emb.astype(np.float64)
    for l in range(m.n_layers):
        taps = {}
        x32 = x_in.astype(np.float32)                      # teacher forcing: the oracle's residual, as fp32
        ref = O.encode(blob, lay, m, x32, tl, w.grid_h, w.grid_w, layer_begin=l, layer_end=l + 1, taps=taps)
        out = g.encode(x32, tl, w.grid_h, w.grid_w, layer_range=(l, l + 1))
        gt = g.taps(T, w.n_frames)
        for key in ("q", "k", "v", "attn", "act"):
            assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_REL_L2, (cfg_id, l, key)
            assert PM.max_row_rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_ROW_REL_L2, (cfg_id, l, key)
        assert PM.rel_l2(out, ref) <= PM.GATE_LAYER_REL_L2
        assert PM.rel_l2(out - x32, ref - x32) <= PM.GATE_LAYER_UPDATE_REL_L2, (cfg_id, l)
        assert PM.max_row_rel_l2(out - x32, ref - x32) <= PM.GATE_ROW_UPDATE_REL_L2, (cfg_id, l)
        oa = g.encode(x32, tl, w.grid_h, w.grid_w, layer_range=(l, l + 1), stop_after_attn=1)
        assert PM.rel_l2(oa - x32, taps["x_attn"][0] - x32) <= PM.GATE_LAYER_UPDATE_REL_L2
        x_in = ref
    g.close()


# ------------------------------------------------------------------------------- whole stacks
def test_cfg1_full_stack(H, O):
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    ref = O.encode(blob, W.blob_layout(w.model), w.model, emb, tl, 4, 4)
    g = H.GpuTE(w.model, w.n_frames, T, blob)
    out = g.encode(emb, tl, 4, 4)
    _assert_final(PM.stack_metrics(out, ref, emb), "cfg1")
    out_direct = g.encode(emb, tl, 4, 4, use_graph=0)
    assert np.array_equal(out, out_direct)                 # graph replay == direct launches, bitwise
    out_again = g.encode(emb, tl, 4, 4)
    assert np.array_equal(out, out_again)                  # deterministic
    g.close()


@pytest.mark.parametrize("cta_pair,resid_bn,split_k", [(1, 128, 1), (1, 256, 1), (0, 256, 1), (0, 128, 1),
                                                       (0, 256, 0), (0, 128, 0)])
def test_cfg1_every_tiling_mode(H, O, cta_pair, resid_bn, split_k):
    """Force each GEMM tiling (one CTA per tile / CTA pairs / split-K groups, 128- and 256-wide residual tiles)."""
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    ref = O.encode(blob, W.blob_layout(w.model), w.model, emb, tl, 4, 4)
    g = H.GpuTE(w.model, w.n_frames, T, blob, cta_pair=cta_pair, resid_bn=resid_bn, split_k=split_k)
    out = g.encode(emb, tl, 4, 4)
    _assert_final(PM.stack_metrics(out, ref, emb), f"pair={cta_pair} bn={resid_bn} split_k={split_k}")
    assert np.array_equal(out, g.encode(emb, tl, 4, 4))    # deterministic (fixed-order partial sums)
    g.close()


def test_ragged_stack_cta_pairs(H, O):
    """CTA-pair tiles on a ragged batch: 3 M tiles of 256 rows with a ragged tail (T = 593 - 10)."""
    m = W.TINY
    blob = H.cached_blob(m, 1)
    tl = [5, 0, 190, 33, 240, 65]
    gh, gw = 2, 5
    T = len(tl) * gh * gw + sum(tl)
    emb = np.random.default_rng(4).standard_normal((T, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, gh, gw)
    g = H.GpuTE(m, len(tl), T, blob, cta_pair=1)
    _assert_final(PM.stack_metrics(g.encode(emb, tl, gh, gw), ref, emb), "ragged pairs")
    g.close()


def test_cfg1_final_norm(H, O):
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    ref = O.encode(blob, W.blob_layout(w.model), w.model, emb, tl, 4, 4, final_norm=1)
    g = H.GpuTE(w.model, w.n_frames, T, blob, final_norm=1)
    out = g.encode(emb, tl, 4, 4)
    assert PM.rel_l2(out, ref) <= 3e-3
    g.close()


@pytest.mark.parametrize("gains", ["ones"])
def test_cfg1_unit_gains(H, O, gains):
    w = W.get_workload(1)
    blob = W.make_weight_blob(w.model, 1, gains=gains)
    tl = W.make_text_lens(w)
    emb = W.make_embeddings(w, 80)
    ref = O.encode(blob, W.blob_layout(w.model), w.model, emb, tl, 4, 4)
    g = H.GpuTE(w.model, 2, 80, blob)
    _assert_final(PM.stack_metrics(g.encode(emb, tl, 4, 4), ref, emb), "unit gains")
    g.close()


def test_ragged_nonsquare_tiny_stack(H, O):
    """Ragged frames incl. a zero-length text and a 200-token frame (4 attention q-blocks,
    2 M tiles with a ragged tail), non-square grid."""
    m = W.TINY
    blob = H.cached_blob(m, 1)
    tl = [5, 0, 190, 33]
    gh, gw = 2, 5
    T = len(tl) * gh * gw + sum(tl)
    emb = np.random.default_rng(3).standard_normal((T, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, gh, gw)
    g = H.GpuTE(m, len(tl), T, blob)
    out = g.encode(emb, tl, gh, gw)
    _assert_final(PM.stack_metrics(out, ref, emb), "ragged")
    g.close()


@pytest.mark.parametrize("cfg_id,frames", [(3, None), (4, [0, 7, 15]), (5, [1, 8, 31])])
def test_full_28_layer_stacks_sampled_frames(H, O, cfg_id, frames):
    """cfg 3 whole; cfg 4/5 at FULL size in the bench launch configuration, compared on sampled
    frames the oracle computes one by one (frames are independent)."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    g = H.GpuTE(m, w.n_frames, T, blob)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    t = g.taps(T, w.n_frames)
    assert np.array_equal(t["pos"], O.position_ids(tl, w.grid_h, w.grid_w))
    assert np.array_equal(t["cu_seqlens"], O.cu_seqlens(tl, w.grid_h, w.grid_w))
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, frames=frames)
    met = PM.stack_metrics(out, ref, emb, ch)
    print(f"cfg{cfg_id} metrics: {met}  out std={out.std():.2f} min={out.min():.1f} max={out.max():.1f}")
    _assert_final(met, f"cfg{cfg_id}")
    assert np.isfinite(out).all()
    g.close()


def test_cfg3_paper_shaped_outliers(H, O):
    """SURVEY Q16 variant: two near-constant channels at the paper's extremes (+1160 / -854)."""
    w, blob, tl, T, emb, ch = H.workload_inputs(3, outliers="paper")
    m = w.model
    g = H.GpuTE(m, w.n_frames, T, blob)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, frames=[0, 3])
    _assert_final(PM.stack_metrics(out, ref, emb, ch), "cfg3 paper-shaped")
    g.close()


# ------------------------------------------------------------------------ invariants on the GPU
def test_zero_projections_pass_residual_bitwise(H):
    """W_o = W_down = 0 => out == embeds BITWISE, outlier channels included (fp32 residual)."""
    w = W.get_workload(1)
    m = w.model
    lay = W.blob_layout(m)
    blob = H.cached_blob(m, 1).copy()
    for l in range(m.n_layers):
        for name in ("Wo", "Wdown"):
            off, shape = lay[(l, name)]
            blob[off:off + int(np.prod(shape))] = 0
    emb = W.make_embeddings(w, 80, outliers="x1000")
    g = H.GpuTE(m, 2, 80, blob)
    out = g.encode(emb, [24, 24], 4, 4)
    assert np.array_equal(out, emb)
    g.close()


def test_frame_independence_permutation_causality_bitwise(H):
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    g = H.GpuTE(w.model, 4, 256, blob)
    out = g.encode(emb, tl, 4, 4)
    solo = g.encode(emb[40:], tl[1:], 4, 4)
    assert np.array_equal(out[40:], solo)
    perm = g.encode(np.concatenate([emb[40:], emb[:40]]), tl[::-1], 4, 4)
    assert np.array_equal(perm[:40], out[40:]) and np.array_equal(perm[40:], out[:40])
    emb2 = emb.copy()
    emb2[30:40] += 1.0
    out2 = g.encode(emb2, tl, 4, 4)
    assert np.array_equal(out[:30], out2[:30]) and np.array_equal(out[40:], out2[40:])
    assert not np.array_equal(out[30:40], out2[30:40])
    g.close()


def test_single_token_frames(H, O):
    """Degenerate: 1x1 grid, no text -> S_b = 1 -> attention output == v."""
    m = W.TINY
    blob = H.cached_blob(m, 1)
    tl = [0, 0, 0]
    emb = np.random.default_rng(5).standard_normal((3, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, 1, 1)
    g = H.GpuTE(m, 3, 3, blob)
    _assert_final(PM.stack_metrics(g.encode(emb, tl, 1, 1), ref, emb), "S=1")
    g.close()


def test_max_tokens_per_frame(H, O):
    """Maximum frame length (256 tokens): 4 attention q-blocks, all kv blocks used."""
    m = W.TINY.with_layers(1)
    blob = H.cached_blob(m, 1)
    tl = [256 - 16]
    emb = np.random.default_rng(6).standard_normal((256, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, 4, 4)
    g = H.GpuTE(m, 1, 256, blob)
    _assert_final(PM.stack_metrics(g.encode(emb, tl, 4, 4), ref, emb), "S=256")
    g.close()


# --------------------------------------------------------------------- boundary / error behaviour
def test_boundary_errors(H):
    import torch
    import paper_2606_05981_b200 as te
    m = W.TINY
    cfg = te.make_config(m, 2, 128)
    h = te.te_create(cfg, 0)
    e = torch.zeros((80, m.hidden), device="cuda")
    o = torch.zeros_like(e)
    tl = torch.tensor([24, 24], dtype=torch.int32, device="cuda")
    L = te.lib()
    assert L.te_encode(h, 2, 4, 4, e.data_ptr(), tl.data_ptr(), 80, o.data_ptr(), None) == te.TE_ERR_NOT_LOADED
    blob = H.cached_blob(m, 1)
    assert L.te_load_weights(h, blob.ctypes.data, blob.nbytes - 2) == te.TE_ERR_BLOB_SIZE
    te.te_load_weights(h, blob)
    assert te.te_blob_bytes(cfg) == blob.nbytes
    assert L.te_encode(h, 3, 4, 4, e.data_ptr(), tl.data_ptr(), 80, o.data_ptr(), None) == te.TE_ERR_INVALID_ARG
    assert L.te_encode(h, 2, 4, 4, e.data_ptr(), tl.data_ptr(), 500, o.data_ptr(), None) == te.TE_ERR_INVALID_ARG
    assert L.te_encode(h, 2, 4, 4, e.data_ptr(), tl.data_ptr(), 80, e.data_ptr(), None) == te.TE_ERR_INVALID_ARG
    assert L.te_encode(h, 2, 4, 4, None, tl.data_ptr(), 80, o.data_ptr(), None) == te.TE_ERR_INVALID_ARG
    # device-side validation: total_tokens that disagrees with the lengths raises the sticky flag
    te.te_encode(h, 2, 4, 4, e, tl, 79, o)
    assert te.te_query_async_error(h) == te.TE_ERR_DEVICE_CHECK
    assert te.te_query_async_error(h) == te.TE_OK
    bad = torch.tensor([-1, 49], dtype=torch.int32, device="cuda")
    te.te_encode(h, 2, 4, 4, e, bad, 80, o)
    assert te.te_query_async_error(h) == te.TE_ERR_DEVICE_CHECK
    te.te_encode(h, 2, 4, 4, e, tl, 80, o)
    assert te.te_query_async_error(h) == te.TE_OK
    bad_cfg = te.make_config(W.TEModelConfig(1, 256, 4, 2, 32, 768, (4, 6, 6)), 2, 128)
    hh = te.c_void_p()
    assert L.te_create(te.byref(bad_cfg), 0, te.byref(hh)) == te.TE_ERR_UNSUPPORTED
    te.te_destroy(h)


def test_encode_is_async_no_sync_and_counts_launches(H):
    """te_encode must not synchronise: after the call returns, the stream still has work queued
    behind a long-running blocker kernel placed before it."""
    import torch
    import paper_2606_05981_b200 as te
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    g = H.GpuTE(w.model, 2, 80, blob)
    g.encode(emb, tl, 4, 4)                                # warm: graph captured
    e, tld, out = g._keep
    st = torch.cuda.Stream()
    n0 = te.te_kernel_launches(g.enc.h)
    with torch.cuda.stream(st):
        torch.cuda._sleep(400_000_000)                     # ~0.2 s of device spin ahead of us
        te.te_encode(g.enc.h, 2, 4, 4, e, tld, 80, out, st.cuda_stream)
        done_at_return = st.query()
    st.synchronize()
    assert not done_at_return
    assert te.te_kernel_launches(g.enc.h) - n0 == 2 + 5 * w.model.n_layers   # refresh + prep + 5 per layer
    g.close()


def test_host_path_matches_device_path(H):
    import torch
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    g = H.GpuTE(w.model, 2, 80, blob)
    out = g.encode(emb, tl, 4, 4)
    eh = torch.from_numpy(emb).pin_memory()
    oh = torch.empty_like(eh).pin_memory()
    g.enc.encode_host(2, 4, 4, eh, np.asarray(tl, dtype=np.int32), oh)
    assert np.array_equal(oh.numpy(), out)
    g.close()


# ------------------------------------------------- interleaved M-RoPE sections
@pytest.mark.parametrize("cfg_id", [1, 2])
def test_interleaved_mrope(H, O, cfg_id):
    """Round-robin t,h,w frequency pairs: rotary table against the oracle's (abs err <= 1e-5), whole stack
    within the gates, and different from the contiguous layout."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model.replace(rope_interleaved=True)
    taps = {}
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, taps=taps)
    g = H.GpuTE(m, w.n_frames, T, blob)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    t = g.taps(T, w.n_frames)
    assert np.max(np.abs(t["cos"] - taps["cos"])) <= PM.GATE_COSSIN_ABS
    assert np.max(np.abs(t["sin"] - taps["sin"])) <= PM.GATE_COSSIN_ABS
    _assert_final(PM.stack_metrics(out, ref, emb), f"interleaved cfg{cfg_id}")
    base = O.encode(blob, W.blob_layout(w.model), w.model, emb, tl, w.grid_h, w.grid_w)
    assert PM.rel_l2(out - emb, base - emb) > 10 * PM.rel_l2(out - emb, ref - emb)   # the layout is visible
    g.close()


# ------------------------------------------- shared text prefix with K/V reuse
def _with_prefix(pre, emb, cu):
    return np.concatenate([np.concatenate([pre, emb[cu[b]:cu[b + 1]]]) for b in range(len(cu) - 1)])


def _strip_prefix(full, P, cu):
    return np.concatenate([full[cu[b] + (b + 1) * P: cu[b + 1] + (b + 1) * P] for b in range(len(cu) - 1)])


@pytest.mark.parametrize("attn_impl", [1, 0])
@pytest.mark.parametrize("cfg_id,P", [(1, 7), (1, 64), (2, 80)])
def test_prefix_kv_reuse_matches_full_recompute(H, O, cfg_id, P, attn_impl):
    """te_encode_prefix once, then te_encode on the frames' own tokens only == the oracle run on the full
    [prefix | grid | text] sequences of every frame (ids continue through the prefix); the prefix rows
    equal the oracle's prefix rows; removing the prefix restores the base path bitwise."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    pre = np.random.default_rng(11 + P).standard_normal((P, m.hidden)).astype(np.float32)
    cu = O.cu_seqlens(tl, w.grid_h, w.grid_w)
    full = _with_prefix(pre, emb, cu)
    ref_full = O.encode(blob, W.blob_layout(m), m, full, tl, w.grid_h, w.grid_w, prefix_len=P)
    ref = _strip_prefix(ref_full, P, cu)
    # attn_impl 1: tcgen05 kernel twice per layer (frame keys, then prefix keys merged through the row
    # statistics); 0: streaming mma.sync kernel over [cached prefix keys | own keys]
    g = H.GpuTE(m, w.n_frames, T, blob, max_prefix_tokens=max(P, 1), attn_impl=attn_impl)
    base = g.encode(emb, tl, w.grid_h, w.grid_w)
    pre_out = g.encode_prefix(pre)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    pos = g.tap(g.te.TE_TAP_POS, (3, T), np.int32)
    want_pos = _strip_prefix(O.position_ids(tl, w.grid_h, w.grid_w, prefix_len=P).T, P, cu).T
    assert np.array_equal(pos, want_pos)
    _assert_final(PM.stack_metrics(out, ref, emb), f"prefix cfg{cfg_id} P={P}")
    _assert_final(PM.stack_metrics(pre_out, ref_full[:P], pre), "prefix rows")
    assert PM.rel_l2(out - emb, base - emb) > 10 * PM.rel_l2(out - emb, ref - emb)   # the prefix is visible
    assert np.array_equal(out, g.encode(emb, tl, w.grid_h, w.grid_w, use_graph=0))
    g.encode_prefix(np.zeros((0, m.hidden), dtype=np.float32))
    assert np.array_equal(g.encode(emb, tl, w.grid_h, w.grid_w), base)
    g.close()


def test_prefix_28_layers_ragged_sampled_frames(H, O):
    """Full depth, ragged batch (cfg 5 lengths, first 12 frames) behind an 80-token prefix:
    S_b + P reaches 240 keys; sampled frames against the oracle's full recompute."""
    w, blob, tl, T, emb, ch = H.workload_inputs(5)
    m = w.model
    B = 12
    tl = tl[:B]
    cu = O.cu_seqlens(tl, w.grid_h, w.grid_w)
    T = int(cu[-1])
    emb = emb[:T]
    P = 80
    pre = np.random.default_rng(5).standard_normal((P, m.hidden)).astype(np.float32)
    g = H.GpuTE(m, B, T, blob, max_prefix_tokens=P)
    g.encode_prefix(pre, want_out=False)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    assert np.isfinite(out).all()
    for b in (0, 7, 11):
        fe = np.concatenate([pre, emb[cu[b]:cu[b + 1]]])
        ref = O.encode(blob, W.blob_layout(m), m, fe, [tl[b]], w.grid_h, w.grid_w, prefix_len=P)[P:]
        met = PM.stack_metrics(out[cu[b]:cu[b + 1]], ref, emb[cu[b]:cu[b + 1]], ch)
        print(f"prefix cfg5 frame {b}: {met}")
        _assert_final(met, f"prefix 28L frame {b}")
    g.close()


def test_pipelined_host_path_matches_blocking_call(H):
    """te_encode_host_submit / _wait with two batches in flight == te_encode_host, bitwise; a third submit
    without a wait is refused."""
    import torch
    import paper_2606_05981_b200 as te
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    g = H.GpuTE(w.model, w.n_frames, T, blob)
    embs = [emb, (emb * 0.5 + 0.25).astype(np.float32), emb[::-1].copy()]
    want = []
    for e in embs:
        o = np.empty_like(e)
        g.enc.encode_host(w.n_frames, w.grid_h, w.grid_w, e, tl, o)
        want.append(o)
    ins = [torch.from_numpy(e).pin_memory() for e in embs]
    outs = [torch.empty_like(i).pin_memory() for i in ins]
    s0 = g.enc.encode_host_submit(w.n_frames, w.grid_h, w.grid_w, ins[0], tl, outs[0])
    s1 = g.enc.encode_host_submit(w.n_frames, w.grid_h, w.grid_w, ins[1], tl, outs[1])
    assert {s0, s1} == {0, 1}
    with pytest.raises(te.TEError):
        g.enc.encode_host_submit(w.n_frames, w.grid_h, w.grid_w, ins[2], tl, outs[2])
    g.enc.encode_host_wait(s0)
    s2 = g.enc.encode_host_submit(w.n_frames, w.grid_h, w.grid_w, ins[2], tl, outs[2])
    g.enc.encode_host_wait(s1)
    g.enc.encode_host_wait(s2)
    for o, wnt in zip(outs, want):
        assert np.array_equal(o.numpy(), wnt)
    with pytest.raises(te.TEError):
        g.enc.encode_host_wait(s2)                      # nothing in flight in that slot any more
    g.close()


@pytest.mark.parametrize("T_target", [1, 127, 129, 255, 257, 513, 767, 1023, 1024, 1025, 1500])
def test_token_count_sweep_across_kernel_regimes(H, O, T_target):
    """Tiny stack at token counts on both sides of every dispatch threshold (one row block / split-K groups /
    CTA pairs at 1024, ragged last row block, 128-wide gate/up tiles): each regime against the oracle."""
    m = W.TINY
    blob = H.cached_blob(m, 1)
    gh, gw = 1, 1
    tl, left = [], T_target
    rng = np.random.default_rng(T_target)
    while left > 0:                                   # frames of 1 visual + up to 254 text tokens
        s = int(min(left, rng.integers(1, 256)))
        tl.append(s - 1)
        left -= s
    T = len(tl) + sum(tl)
    assert T == T_target
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, gh, gw)
    g = H.GpuTE(m, len(tl), T, blob)
    out = g.encode(emb, tl, gh, gw)
    _assert_final(PM.stack_metrics(out, ref, emb), f"T={T}")
    assert np.array_equal(g.tap(g.te.TE_TAP_CU_SEQLENS, (len(tl) + 1,), np.int32), O.cu_seqlens(tl, gh, gw))
    g.close()


@pytest.mark.parametrize("T_target", [256, 384, 640, 1024, 1280])
def test_full_width_layer_token_sweep(H, O, T_target):
    """One full-width layer (cfg 2 shape) at mid token counts: the per-GEMM choice between split-K groups, one CTA per
    tile and CTA pairs depends on tiles vs SMs (e.g. T = 256: QKV 64 tiles x 2 K-slices, O-proj/down 32 x 4,
    gate/up 96 tiles; T = 640: gate/up on CTA pairs)."""
    w, blob, _, _, _, _ = H.workload_inputs(2)
    m = w.model
    rng = np.random.default_rng(T_target)
    tl, left = [], T_target
    while left > 0:
        s = int(min(left, 64 + rng.integers(1, 192)))
        if s <= 64:
            tl[-1] += s                              # fold a short remainder into the previous frame's text
            left = 0
            break
        tl.append(s - 64)
        left -= s
    tl = [int(t) for t in tl]
    assert all(64 + t <= 256 for t in tl[:-1])
    if 64 + tl[-1] > 256:                            # keep every frame within max_tokens_per_frame
        extra = 64 + tl[-1] - 256
        tl[-1] -= extra
        tl.append(max(0, extra - 64))
    T = 64 * len(tl) + sum(tl)
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, 8, 8)
    g = H.GpuTE(m, len(tl), T, blob)
    out = g.encode(emb, tl, 8, 8)
    _assert_final(PM.stack_metrics(out, ref, emb), f"full-width T={T}")
    g.close()


@pytest.mark.parametrize("hq,hkv,dh", [(4, 4, 64), (8, 2, 64), (8, 1, 64), (6, 2, 64), (2, 2, 128), (6, 1, 128)])
def test_gqa_group_sizes(H, O, hq, hkv, dh):
    """Query-group sizes G = Hq/Hkv in {1, 2, 3, 4, 6, 8}: the tcgen05 attention kernel stacks G heads into a query
    tile when G is a power of two <= 8; other G (3, 6) run on the streaming kernel.  Small 2-layer stacks vs oracle."""
    hidden = 256
    sec = (8, 12, 12) if dh == 64 else (16, 24, 24)
    m = W.TEModelConfig(n_layers=2, hidden=hidden, n_q_heads=hq, n_kv_heads=hkv, head_dim=dh, ffn=512,
                        rope_sections=sec)
    if ((hq + 2 * hkv) * dh) % 128 != 0:
        pytest.skip("fused QKV width must be a multiple of 128")
    blob = W.make_weight_blob(m, 7)
    tl = [30, 0, 201, 77]
    gh, gw = 3, 4
    T = len(tl) * gh * gw + sum(tl)
    emb = np.random.default_rng(hq * 10 + hkv).standard_normal((T, hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, gh, gw)
    g = H.GpuTE(m, len(tl), T, blob)
    _assert_final(PM.stack_metrics(g.encode(emb, tl, gh, gw), ref, emb), f"Hq={hq} Hkv={hkv} dh={dh}")
    g.close()


def test_many_small_frames(H, O):
    """300 frames of 1-6 tokens: the device-side scan runs over several 32-frame chunks, every attention CTA sees a
    nearly empty frame, frames straddle row-block boundaries."""
    m = W.TINY
    blob = H.cached_blob(m, 1)
    rng = np.random.default_rng(12)
    tl = [int(t) for t in rng.integers(0, 6, size=300)]
    gh, gw = 1, 1
    T = len(tl) + sum(tl)
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, gh, gw)
    g = H.GpuTE(m, len(tl), T, blob)
    out = g.encode(emb, tl, gh, gw)
    assert np.array_equal(g.tap(g.te.TE_TAP_POS, (3, T), np.int32), O.position_ids(tl, gh, gw))
    assert np.array_equal(g.tap(g.te.TE_TAP_CU_SEQLENS, (len(tl) + 1,), np.int32), O.cu_seqlens(tl, gh, gw))
    _assert_final(PM.stack_metrics(out, ref, emb), "300 frames")
    g.close()


@pytest.mark.parametrize("n_tiles", [2, 3, 5, 8])
def test_wide_residual_tiles(H, O, n_tiles):
    """O-proj / down as one wave of wide CTA-pair tiles: forced tile counts whose widths do and do not divide the hidden
    size (a partly and a completely out-of-range last tile), ragged last row-pair block."""
    m = W.TINY
    blob = H.cached_blob(m, 1)
    tl = [5, 0, 190, 33, 240, 65]
    gh, gw = 2, 5
    T = len(tl) * gh * gw + sum(tl)
    emb = np.random.default_rng(4).standard_normal((T, m.hidden)).astype(np.float32)
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, gh, gw)
    g = H.GpuTE(m, len(tl), T, blob, cta_pair=1, resid_wide=n_tiles)
    out = g.encode(emb, tl, gh, gw)
    _assert_final(PM.stack_metrics(out, ref, emb), f"wide residual tiles n={n_tiles}")
    assert np.array_equal(out, g.encode(emb, tl, gh, gw))
    g.close()


def test_two_handles_share_the_gpu(H):
    """Two encoders running their split-K (spinning) kernels on two streams at the same time: cooperative launches
    keep each group co-resident, so the runs interleave instead of deadlocking, and the results are unchanged."""
    import torch
    w, blob, tl, T, emb, ch = H.workload_inputs(2)
    ga = H.GpuTE(w.model, w.n_frames, T, blob)
    gb = H.GpuTE(w.model, w.n_frames, T, blob)
    want = ga.encode(emb, tl, w.grid_h, w.grid_w)
    e = torch.from_numpy(emb).cuda()
    lens = torch.from_numpy(tl).cuda()
    oa, ob = torch.empty_like(e), torch.empty_like(e)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(50):
        ga.enc.encode(w.n_frames, w.grid_h, w.grid_w, e, lens, T, oa, sa.cuda_stream)
        gb.enc.encode(w.n_frames, w.grid_h, w.grid_w, e, lens, T, ob, sb.cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(oa.cpu().numpy(), want) and np.array_equal(ob.cpu().numpy(), want)
    ga.close()
    gb.close()


def test_encode_inside_a_callers_graph_capture(H):
    """The call performs no sync, copy or allocation, so a caller can capture it into a CUDA graph of its own
    (e.g. together with the denoiser step): the library then enqueues its kernels directly into that capture."""
    import torch
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    g = H.GpuTE(w.model, w.n_frames, T, blob)
    want = g.encode(emb, tl, w.grid_h, w.grid_w)
    e = torch.from_numpy(emb).cuda()
    lens = torch.from_numpy(tl).cuda()
    out = torch.zeros_like(e)
    st = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(graph, stream=st):
        g.enc.encode(w.n_frames, w.grid_h, w.grid_w, e, lens, T, out, torch.cuda.current_stream().cuda_stream)
    for _ in range(3):
        out.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), want)
    g.close()


# ------------------------------------------- every row at full size (next #1b)
def _one_layer_all_rows(H, O, w, blob, tl, T, emb, layer, tag):
    """Teacher-forced ONE layer over ALL rows through the default dispatch: taps and the update, per token row."""
    m = w.model
    g = H.GpuTE(m, w.n_frames, T, blob)
    taps = {}
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, layer_begin=layer, layer_end=layer + 1,
                   taps=taps)
    out = g.encode(emb, tl, w.grid_h, w.grid_w, layer_range=(layer, layer + 1))
    gt = g.taps(T, w.n_frames)
    info = g.te.te_dispatch_info(g.enc.h)
    for key in ("q", "k", "v", "attn", "act"):
        assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_REL_L2, (tag, key)
        assert PM.max_row_rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_ROW_REL_L2, (tag, key)
    e64 = emb.astype(np.float64)
    assert PM.rel_l2(out - e64, ref - e64) <= PM.GATE_LAYER_UPDATE_REL_L2, tag
    rows = PM.row_rel_l2(out - e64, ref - e64)
    assert rows.max() <= PM.GATE_ROW_UPDATE_REL_L2, (tag, int(rows.argmax()), float(rows.max()))
    oa = g.encode(emb, tl, w.grid_h, w.grid_w, layer_range=(layer, layer + 1), stop_after_attn=1)
    assert PM.max_row_rel_l2(oa - e64, taps["x_attn"][0] - e64) <= PM.GATE_ROW_UPDATE_REL_L2, tag
    print(f"{tag}: dispatch {info}; max row update rel-L2 {rows.max():.2e} (row {rows.argmax()})")
    g.close()
    return info


@pytest.mark.parametrize("cfg_id,layer", [(4, 0), (4, 27), (5, 13)])
def test_one_layer_every_row_full_size(H, O, cfg_id, layer):
    """cfg 4 (T = 3072: CTA pairs + 6 x 352 wide residual tiles) and cfg 5 (ragged T: 4 x 512) at FULL size: one
    teacher-forced layer compared with the oracle on EVERY row — all 12-15 row-pair blocks, every wide residual tile,
    every attention (frame, head) — not on sampled frames."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    info = _one_layer_all_rows(H, O, w, blob, tl, T, emb, layer, f"cfg{cfg_id} layer {layer}")
    assert info["oproj"].startswith("te_gemm_wide_kernel") and info["qkv"].startswith("te_gemm2_kernel")


def test_one_layer_every_row_mid_batch(H, O):
    """cfg 3 (T = 512): split-K groups + the one-wave wide SwiGLU tiles over the interleaved gate/up weights."""
    w, blob, tl, T, emb, ch = H.workload_inputs(3)
    info = _one_layer_all_rows(H, O, w, blob, tl, T, emb, 5, "cfg3 layer 5")
    assert info["gateup"].startswith("te_gemm_wide_kernel<3>") and info["qkv"].startswith("te_gemmk_kernel")


@pytest.mark.parametrize("cfg_id", [4, 5])
def test_identical_frames_cover_every_row_of_the_28_layer_stack(H, O, cfg_id):
    """Full depth, full size, EVERY row: all frames get the same embeddings (cut to their own length), so by
    causality frame b's rows must equal the first S_b rows of the longest frame BITWISE — whatever row block, wide
    tile or attention CTA they land in — and the longest frame is compared with the oracle."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    cu = O.cu_seqlens(tl, w.grid_h, w.grid_w)
    b_long = int(np.argmax(np.diff(cu)))
    base = emb[cu[b_long]:cu[b_long + 1]]
    same = np.concatenate([base[: cu[b + 1] - cu[b]] for b in range(w.n_frames)])
    g = H.GpuTE(m, w.n_frames, T, blob)
    out = g.encode(same, tl, w.grid_h, w.grid_w)
    want = out[cu[b_long]:cu[b_long + 1]]
    for b in range(w.n_frames):
        assert np.array_equal(out[cu[b]:cu[b + 1]], want[: cu[b + 1] - cu[b]]), f"frame {b} differs from frame {b_long}"
    ref = O.encode(blob, W.blob_layout(m), m, base, [tl[b_long]], w.grid_h, w.grid_w)
    met = PM.stack_metrics(want, ref, base, ch)
    print(f"cfg{cfg_id} identical frames: {met}")
    _assert_final(met, f"cfg{cfg_id} identical frames")
    g.close()


# ------------------------------------------------------- graph reuse
def test_graph_reuse_ragged_lengths_and_changing_buffers(H, O):
    """200 calls with fresh random ragged lengths and alternating buffers: a graph is captured once per shape class
    (row-block bucket of the token count), never per call or per pointer; the last call is compared with the oracle."""
    import torch
    import paper_2606_05981_b200 as te
    m = W.TINY
    blob = H.cached_blob(m, 1)
    B, gh, gw = 12, 2, 3
    cap = B * 256
    g = H.GpuTE(m, B, cap, blob)
    rng = np.random.default_rng(99)
    bufs = [(torch.empty((cap, m.hidden), device="cuda"), torch.empty((cap, m.hidden), device="cuda"),
             torch.empty(B, dtype=torch.int32, device="cuda")) for _ in range(3)]
    te.te_debug_set_range(g.enc.h, 0, m.n_layers, 0)
    buckets = set()
    c0 = te.te_graph_captures(g.enc.h)
    last = None
    for i in range(200):
        tl = rng.integers(60, 140, size=B).astype(np.int32)
        T = int(B * gh * gw + tl.sum())
        buckets.add((T + 255) // 256 if (T + 127) // 128 * 128 >= 1024 else -((T + 127) // 128))
        e, o, l = bufs[i % 3]
        emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
        e[:T].copy_(torch.from_numpy(emb))
        l.copy_(torch.from_numpy(tl))
        g.enc.encode(B, gh, gw, e, l, T, o)
        last = (emb, tl, T, o)
    torch.cuda.synchronize()
    assert te.te_query_async_error(g.enc.h) == te.TE_OK
    n_cap = te.te_graph_captures(g.enc.h) - c0
    assert n_cap == len(buckets) and n_cap <= 6, (n_cap, sorted(buckets))
    emb, tl, T, o = last
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, gh, gw)
    _assert_final(PM.stack_metrics(o[:T].cpu().numpy(), ref, emb), "graph reuse, last call")
    # same bucket, different T and pointers: identical to a fresh handle's result, bitwise
    g2 = H.GpuTE(m, B, cap, blob)
    assert np.array_equal(g2.encode(emb, tl, gh, gw), o[:T].cpu().numpy())
    g2.close()
    g.close()


def test_stale_rows_of_a_larger_call_do_not_leak(H, O):
    """The activation tensor maps span the whole workspace: after a large call whose rows are NaN-poisoned, a smaller
    call (its last frame's length not a multiple of 16, so the attention tiles read past it) must be unaffected."""
    m = W.TINY
    blob = H.cached_blob(m, 1)
    g = H.GpuTE(m, 4, 1024, blob)
    big = np.full((1000, m.hidden), np.nan, dtype=np.float32)
    g.encode(big, [249, 249, 249, 249], 1, 1)
    tl = [100, 37]
    T = 2 + sum(tl)
    emb = np.random.default_rng(8).standard_normal((T, m.hidden)).astype(np.float32)
    out = g.encode(emb, tl, 1, 1)
    assert np.isfinite(out).all()
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, 1, 1)
    _assert_final(PM.stack_metrics(out, ref, emb), "after a poisoned larger call")
    g.close()


# --------------------------------------------- side stream against a foreign load
@pytest.mark.parametrize("budget", [0, 74])
@pytest.mark.parametrize("case", ["cfg2_split_k", "pairs_T1024"])
def test_side_stream_under_foreign_load_is_bitwise_identical(H, case, budget):
    """The paper's mechanism 1 (Algorithm 1 :118-137): te_encode on a SIDE stream while the main stream
    runs a denoiser-shaped load (library bf16 matmuls), joined by one event.  The result must be bitwise the solo
    result — the cooperative split-K groups (cfg 2) and the CTA-pair kernels (T = 1024) only get delayed.
    budget = 74: the same with the encoder sized for half the SMs (TE_OPT_SM_BUDGET), the arrangement that lets the
    foreign load actually run beside it."""
    import torch
    import paper_2606_05981_b200 as te
    w, blob, tl, T, emb, ch = H.workload_inputs(2)
    m = w.model
    if case == "pairs_T1024":
        tl = np.full(8, 64, dtype=np.int32)
        T = 8 * 128
        emb = np.random.default_rng(17).standard_normal((T, m.hidden)).astype(np.float32)
    B = len(tl)
    g = H.GpuTE(m, B, T, blob)
    te.te_set_option(g.enc.h, te.TE_OPT_SM_BUDGET, budget)
    solo = g.encode(emb, tl, w.grid_h, w.grid_w)
    e, lens, out = g._keep
    a = torch.randn(4096, 4096, device="cuda", dtype=torch.bfloat16)
    b = torch.randn(4096, 4096, device="cuda", dtype=torch.bfloat16)
    c = torch.empty_like(a)
    side = torch.cuda.Stream()
    main = torch.cuda.current_stream()
    for _ in range(5):
        out.zero_()
        ev0, ev = torch.cuda.Event(), torch.cuda.Event()
        ev0.record(main)
        side.wait_event(ev0)
        with torch.cuda.stream(side):
            for _ in range(4):
                te.te_encode(g.enc.h, B, w.grid_h, w.grid_w, e, lens, T, out, side.cuda_stream)
            ev.record(side)
        for _ in range(12):
            torch.matmul(a, b, out=c)                   # the foreign load, concurrently on the main stream
        main.wait_event(ev)                             # the single cross-stream event of Algorithm 1
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), solo)
    assert te.te_query_async_error(g.enc.h) == te.TE_OK
    g.close()


@pytest.mark.parametrize("budget", [74, 112, 16])
def test_sm_budget_changes_the_grids_not_the_results(H, O, budget):
    """TE_OPT_SM_BUDGET (te.h): every GEMM grid and dispatch decision sized for `budget` SMs.  One full-width layer
    against the fp64 oracle in the split-K regime (T = 128), the CTA-pair regime (T = 1024) against the full-GPU run of
    the same handle, both bitwise repeatable; out-of-range budgets are refused."""
    import paper_2606_05981_b200 as te
    w, blob, tl, T, emb, ch = H.workload_inputs(2)
    m = w.model
    ref = O.encode(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w)
    g = H.GpuTE(m, 8, 1024, blob)
    full_info = None
    tl8 = np.full(8, 64, dtype=np.int32)
    emb8 = np.random.default_rng(17).standard_normal((1024, m.hidden)).astype(np.float32)
    full8 = g.encode(emb8, tl8, w.grid_h, w.grid_w)
    full_info = te.te_dispatch_info(g.enc.h)
    te.te_set_option(g.enc.h, te.TE_OPT_SM_BUDGET, budget)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    _assert_final(PM.stack_metrics(out, ref, emb), f"sm budget {budget}, T=128")
    assert np.array_equal(out, g.encode(emb, tl, w.grid_h, w.grid_w))
    out8 = g.encode(emb8, tl8, w.grid_h, w.grid_w)
    mm = PM.stack_metrics(out8, full8, emb8)
    assert mm["update_rel_l2"] <= PM.GATE_UPDATE_REL_L2 and mm["max_row_update_rel_l2"] <= PM.GATE_ROW_UPDATE_REL_L2, mm
    assert np.array_equal(out8, g.encode(emb8, tl8, w.grid_h, w.grid_w))
    if budget == 74:   # 37 CTA pairs: the residual GEMMs' 128-wide tiles would need two waves -> one wave of wide tiles
        assert te.te_dispatch_info(g.enc.h) != full_info         # (at 16 or 112 SMs only the grids shrink, not the kernels)
    assert te.te_query_async_error(g.enc.h) == te.TE_OK
    for bad in (1, 15, 100000, -3):
        assert te.lib().te_set_option(g.enc.h, te.TE_OPT_SM_BUDGET, bad) == te.TE_ERR_INVALID_ARG
    te.te_set_option(g.enc.h, te.TE_OPT_SM_BUDGET, 0)             # back to the whole GPU: bitwise the first result
    assert np.array_equal(g.encode(emb8, tl8, w.grid_h, w.grid_w), full8)
    g.close()


def test_sm_budget_28_layers(H):
    """The 28-layer stack at B = 4 under a 74-SM budget: close to the full-GPU run at the stack gates, and repeatable."""
    import paper_2606_05981_b200 as te
    w, blob, tl, T, emb, ch = H.workload_inputs(3)
    g = H.GpuTE(w.model, w.n_frames, T, blob)
    full = g.encode(emb, tl, w.grid_h, w.grid_w)
    te.te_set_option(g.enc.h, te.TE_OPT_SM_BUDGET, 74)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    assert np.array_equal(out, g.encode(emb, tl, w.grid_h, w.grid_w))
    _assert_final(PM.stack_metrics(out, full, emb), "sm budget 74, cfg 3")
    g.close()


# ------------------------------------------------------------------ runtime hygiene
def test_two_handles_on_two_host_threads(H):
    """Launch state is per handle: two handles with DIFFERENT options driven from two host threads at once."""
    import threading
    import torch
    w, blob, tl, T, emb, ch = H.workload_inputs(2)
    ga = H.GpuTE(w.model, w.n_frames, T, blob)                      # split-K groups (cooperative launches)
    gb = H.GpuTE(w.model, w.n_frames, T, blob, split_k=0)           # one CTA per tile
    want_a = ga.encode(emb, tl, w.grid_h, w.grid_w)
    want_b = gb.encode(emb, tl, w.grid_h, w.grid_w)
    e = torch.from_numpy(emb).cuda()
    lens = torch.from_numpy(tl).cuda()
    outs = {"a": torch.empty_like(e), "b": torch.empty_like(e)}
    errs = []

    def drive(g, key):
        try:
            st = torch.cuda.Stream()
            for _ in range(100):
                g.enc.encode(w.n_frames, w.grid_h, w.grid_w, e, lens, T, outs[key], st.cuda_stream)
            st.synchronize()
        except Exception as ex:                       # noqa: BLE001
            errs.append(ex)

    ts = [threading.Thread(target=drive, args=(ga, "a")), threading.Thread(target=drive, args=(gb, "b"))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    torch.cuda.synchronize()
    assert not errs, errs
    assert np.array_equal(outs["a"].cpu().numpy(), want_a) and np.array_equal(outs["b"].cpu().numpy(), want_b)
    ga.close()
    gb.close()


def test_create_destroy_does_not_leak(H):
    """100 create / load / prefix / encode / destroy cycles: free device memory returns to where it started."""
    import torch
    m = W.TINY
    blob = H.cached_blob(m, 1)
    emb = np.random.default_rng(2).standard_normal((80, m.hidden)).astype(np.float32)
    pre = np.random.default_rng(3).standard_normal((16, m.hidden)).astype(np.float32)

    def cycle():
        g = H.GpuTE(m, 2, 80, blob, max_prefix_tokens=16)
        g.encode_prefix(pre, want_out=False)
        g.encode(emb, [24, 24], 4, 4)
        g._keep = None
        g.close()

    cycle()
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(100):
        cycle()
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < (8 << 20), (free0, free1)     # (allocator granularity; one leaked cycle would be > 3 MB x 100)


def test_host_path_refuses_a_frame_longer_than_the_capacity(H):
    import paper_2606_05981_b200 as te
    m = W.TINY
    blob = H.cached_blob(m, 1)
    g = H.GpuTE(m, 2, 512, blob)
    emb = np.zeros((16 + 250 + 16 + 10, m.hidden), dtype=np.float32)
    out = np.empty_like(emb)
    with pytest.raises(te.TEError) as ei:
        g.enc.encode_host(2, 4, 4, emb, np.asarray([250, 10], dtype=np.int32), out)     # 16 + 250 > 256
    assert ei.value.code == te.TE_ERR_INVALID_ARG
    g.close()


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_shape_sweep_all_dtypes(H, O, seed):
    """Seeded random calls on ONE handle per operand type (bf16 / MXFP8 / MXFP4 weights): 1-40 frames, grids 1x1 .. 8x8,
    text lengths 0 .. 256 - grid (token counts on both sides of the CTA-pair threshold, many graph shape classes,
    shrinking and growing), each against its oracle with the per-row gates; ids bit-exact."""
    from oracle import te_mxfp8 as Q
    import paper_2606_05981_b200 as te
    m = W.TINY
    blob = H.cached_blob(m, 1)
    lay = W.blob_layout(m)
    rng = np.random.default_rng(seed)
    encs = {dt: H.GpuTE(m, 40, 4096, blob, weight_dtype=dt) for dt in (0, 1, 2)}
    for case in range(10):
        dt = int(rng.integers(0, 3))
        B = int(rng.integers(1, 41))
        gh, gw = int(rng.integers(1, 9)), int(rng.integers(1, 9))
        tl = rng.integers(0, 257 - gh * gw, size=B).astype(np.int32)
        while B * gh * gw + int(tl.sum()) > 4000:
            tl = (tl // 2).astype(np.int32)
        T = B * gh * gw + int(tl.sum())
        emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
        g = encs[dt]
        out = g.encode(emb, tl, gh, gw)
        if dt == 0:
            mm = PM.stack_metrics(out, O.encode(blob, lay, m, emb, tl, gh, gw), emb)
            assert PM.passes_final_gates(mm), (case, B, gh, gw, T, mm)
        else:
            mm = PM.stack_metrics(out, Q.encode_mxfp8(blob, lay, m, emb, tl, gh, gw, fp4_weights=(dt == 2)), emb)
            assert PM.passes_mx_gates(mm), (case, dt, B, gh, gw, T, mm)
        assert np.array_equal(g.tap(te.TE_TAP_POS, (3, T), np.int32), O.position_ids(tl, gh, gw))
        assert te.te_query_async_error(g.enc.h) == te.TE_OK
    for g in encs.values():
        g.close()


# ------------------------------------------------------------------- device-wide L2 settings
def _persisting_l2_limit():
    """cudaDeviceGetLimit(cudaLimitPersistingL2CacheSize) of the current device, through the runtime torch loaded (the
    limit belongs to the device's primary context, which the library shares)."""
    import ctypes
    import glob
    import os
    import torch
    cands = glob.glob(os.path.join(os.path.dirname(torch.__file__), "..", "nvidia", "cuda_runtime", "lib", "libcudart.so*"))
    cands += ["libcudart.so.12", "libcudart.so"]
    for c in cands:
        try:
            rt = ctypes.CDLL(c)
            break
        except OSError:
            continue
    else:
        pytest.skip("no libcudart to query the limit with")
    v = ctypes.c_size_t(0)
    assert rt.cudaDeviceGetLimit(ctypes.byref(v), 6) == 0        # cudaLimitPersistingL2CacheSize = 0x06
    return v.value


def test_persisting_l2_limit_is_shared_by_handles_and_restored_by_the_last(H):
    """Two live handles (the decoder + vision-tower pairing): the device-wide persisting-L2 limit is raised once, stays
    up when the handle that raised it is destroyed FIRST, still serves the survivor (same bits), and returns to the
    value found before the first handle only when the last one goes — whatever the destruction order."""
    import torch
    w, blob, tl, T, emb, ch = H.workload_inputs(2)
    torch.cuda.synchronize()
    before = _persisting_l2_limit()
    a = H.GpuTE(w.model, len(tl), T, blob)
    ref = a.encode(emb, tl, w.grid_h, w.grid_w)
    raised = _persisting_l2_limit()
    assert raised >= min(T, 128) * w.model.hidden * 4 and raised >= before
    b = H.GpuTE(w.model, len(tl), T, blob)
    assert np.array_equal(b.encode(emb, tl, w.grid_h, w.grid_w), ref)
    assert _persisting_l2_limit() == raised
    a.close()                                                    # the one that raised it goes first
    assert _persisting_l2_limit() == raised
    assert np.array_equal(b.encode(emb, tl, w.grid_h, w.grid_w), ref)
    b.close()
    assert _persisting_l2_limit() == before
    c = H.GpuTE(w.model, len(tl), T, blob)                       # and the cycle starts clean again
    assert np.array_equal(c.encode(emb, tl, w.grid_h, w.grid_w), ref)
    c.close()
    assert _persisting_l2_limit() == before


def test_residual_larger_than_the_access_policy_window(H):
    """72 frames x 256 tokens x 2048 x 4 B = 151 MB of fp32 residual: more than accessPolicyMaxWindowSize.  The L2 window
    must shrink to what the device allows instead of making every launch fail; results equal the no-window run bitwise."""
    import torch
    import paper_2606_05981_b200 as te
    w = W.get_workload(2)
    m = w.model
    B, text = 72, 192
    T = B * (w.grid_h * w.grid_w + text)
    assert T * m.hidden * 4 > torch.cuda.get_device_properties(0).L2_cache_size
    blob = H.cached_blob(m, w.seed_weights)
    emb = np.random.default_rng(5).standard_normal((T, m.hidden)).astype(np.float32)
    tl = np.full(B, text, dtype=np.int32)
    g = H.GpuTE(m, B, T, blob)
    got = g.encode(emb, tl, w.grid_h, w.grid_w)                  # default options: window on
    assert te.te_query_async_error(g.enc.h) == te.TE_OK
    te.te_set_option(g.enc.h, te.TE_OPT_L2_RESIDUAL, 0)
    plain = g.encode(emb, tl, w.grid_h, w.grid_w)
    g.close()
    assert np.isfinite(got).all() and np.array_equal(got, plain)
    # frames are independent and identical in shape: frame 0 of this batch == the same frame encoded alone
    S = w.grid_h * w.grid_w + text
    g1 = H.GpuTE(m, 1, S, blob)
    alone = g1.encode(emb[:S], tl[:1], w.grid_h, w.grid_w)
    g1.close()
    assert PM.rel_l2(got[:S], alone) < 1e-3
