"""`-m gpu` parity tests of the block-scaled FP8 variant (te_config.weight_dtype = 1) against
the MXFP8 oracle (oracle/te_mxfp8.py, readings Q24-Q27 of DESIGN.md §3).  Integer work (the quantiser's codes and
scales) is compared bit-exactly; the block-scaled GEMM alone to fp32-accumulation accuracy; stacks within the gates
tests/parity_metrics.py derives for two 8-bit pipelines."""
import numpy as np
import pytest

import workloads as W
import parity_metrics as PM

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Q():
    from oracle import te_mxfp8
    return te_mxfp8


@pytest.fixture(scope="module")
def O():
    from oracle import te_oracle
    return te_oracle


@pytest.fixture(scope="module")
def H():
    import gpu_helpers
    return gpu_helpers


def _assert_mx(m, tag="", deep=False):
    assert PM.passes_mx_gates(m, deep), (tag, m)
    assert m["cos_sim"] > 0.999, (tag, m)


def _bf16_matrix(rng, rows, K, outliers=True):
    x = rng.standard_normal((rows, K)).astype(np.float32)
    if outliers and rows >= 8:
        x[:, 5] *= 1000.0                      # an outlier channel: its 32-block gets a large scale, the others do not
        x[::7, 40:72] = 0.0                    # an all-zero block
        x[3, 100] = 448.0 * 2.0 ** 5           # exactly on the 1.75 * 2^n boundary of the scale rule
        x[4, 110] = 2.0 ** -30                 # deep in the subnormal range of its block
    return W.f32_to_bf16_bits(x)


@pytest.mark.parametrize("rows,K", [(128, 128), (300, 256), (517, 2048), (2048, 6144)])
def test_quantiser_codes_and_scales_bit_exact(H, Q, rows, K):
    """The device quantiser (weights at te_load_weights; same device functions in the epilogues) against the oracle's:
    E4M3 codes and E8M0 scales are integers -> bit-exact."""
    import torch
    import paper_2606_05981_b200 as te
    bits = _bf16_matrix(np.random.default_rng(rows + K), rows, K)
    src = torch.from_numpy(bits.view(np.int16)).cuda()
    rb = (rows + 127) // 128
    codes = torch.zeros((rows, K), dtype=torch.uint8, device="cuda")
    sft = torch.full((rb, K // 128, 512), 0xEE, dtype=torch.uint8, device="cuda")
    te.te_debug_mx_quantise(0, src, rows, K, codes, sft)
    want_codes, want_sf = Q.quantise(H.bf16_bits_to_f64(bits).reshape(rows, K))
    got_sf = H.untile_scales(sft.cpu().numpy(), rows, K)
    assert np.array_equal(got_sf, want_sf)
    got = codes.cpu().numpy()
    # +0 and -0 are the same value; everything else must be the same byte
    same = (got == want_codes) | (((got | want_codes) & 0x7F) == 0)
    assert same.all(), np.argwhere(~same)[:5]
    assert np.array_equal(H.mx_dequant(got, got_sf), Q.dequantise(want_codes, want_sf))


@pytest.mark.parametrize("M,N,K,bn", [(128, 128, 128, 128), (256, 256, 128, 256), (1, 128, 256, 128), (300, 512, 256, 128),
                                       (300, 512, 256, 256), (517, 768, 896, 256), (3072, 4096, 2048, 128),
                                       (3072, 4096, 2048, 256), (3072, 2048, 6144, 128), (1500, 1536, 2048, 256)])
def test_gemm_mxfp8_vs_fp64_of_the_dequantised_operands(H, Q, M, N, K, bn):
    """Block-scaled tcgen05 main loop alone (scale tiles -> TMEM, K = 32 MMAs selecting their scale byte): with both
    operands quantised by the (bit-exact) device quantiser the product must equal the fp64 product of the DEQUANTISED
    operands to fp32-accumulation accuracy.  A wrong scale tile, byte or TMEM column shows as an O(1) error."""
    import torch
    import paper_2606_05981_b200 as te
    rng = np.random.default_rng(M * 5 + N + K)
    a = _bf16_matrix(rng, M, K)
    b = W.f32_to_bf16_bits((rng.standard_normal((N, K)) * np.exp(rng.uniform(-3, 3, size=(N, 1)))).astype(np.float32))
    A = Q.fake_quant(H.bf16_bits_to_f64(a).reshape(M, K))
    B = Q.fake_quant(H.bf16_bits_to_f64(b).reshape(N, K))
    ref = A @ B.T
    ad = torch.from_numpy(a.view(np.int16)).cuda()
    bd = torch.from_numpy(b.view(np.int16)).cuda()
    c = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    te.te_debug_gemm_mxfp8(0, ad, bd, c, M, N, K, bn)
    out = c.cpu().numpy()
    assert np.isfinite(out).all()
    assert PM.rel_l2(out, ref) < 1e-5
    scale = np.linalg.norm(A, axis=1)[:, None] * np.linalg.norm(B, axis=1)[None, :]
    assert np.max(np.abs(out - ref) / scale) < 1e-5


def test_cfg1_stack_mxfp8(H, O, Q):
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    ref = Q.encode_mxfp8(blob, W.blob_layout(w.model), w.model, emb, tl, 4, 4)
    g = H.GpuTE(w.model, w.n_frames, T, blob, weight_dtype=1)
    out = g.encode(emb, tl, 4, 4)
    met = PM.stack_metrics(out, ref, emb)
    print("cfg1 mxfp8:", met)
    _assert_mx(met, "cfg1 mxfp8")
    assert np.array_equal(out, g.encode(emb, tl, 4, 4, use_graph=0))           # graph == direct launches
    assert np.array_equal(out, g.encode(emb, tl, 4, 4))                         # deterministic
    plain = O.encode(blob, W.blob_layout(w.model), w.model, emb, tl, 4, 4)
    # the quantised network is a different function: further from the unquantised oracle than from its own
    assert PM.rel_l2(out - emb, plain - emb) > 2 * PM.rel_l2(out - emb, ref - emb)
    info = g.te.te_dispatch_info(g.enc.h)
    assert info["gateup"].startswith("te_gemm8_kernel")
    g.close()


@pytest.mark.parametrize("cfg_id", [1, 2])
def test_layer0_taps_mxfp8(H, Q, cfg_id):
    """Layer 0, teacher-forced: the first GEMM's A operand is quantised from the SAME fp32 values on both sides, so
    q/k/v meet the bf16-class tap gate; the quantised attention / SwiGLU outputs are compared after dequantisation."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    taps = {}
    ref = Q.encode_mxfp8(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, layer_begin=0, layer_end=1, taps=taps)
    g = H.GpuTE(m, w.n_frames, T, blob, weight_dtype=1)
    out = g.encode(emb, tl, w.grid_h, w.grid_w, layer_range=(0, 1))
    gt = g.taps_mx(T)
    for key in ("q", "k", "v"):
        assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_REL_L2, (cfg_id, key, PM.rel_l2(gt[key], taps[key][0]))
        assert PM.max_row_rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_ROW_REL_L2, (cfg_id, key)
    for key in ("attn", "act"):
        assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_MX_TAP_REL_L2, (cfg_id, key, PM.rel_l2(gt[key], taps[key][0]))
    e64 = emb.astype(np.float64)
    assert PM.rel_l2(out - e64, ref - e64) <= PM.GATE_MX_UPDATE_REL_L2
    assert PM.max_row_rel_l2(out - e64, ref - e64) <= PM.GATE_MX_ROW_UPDATE_REL_L2
    g.close()


@pytest.mark.parametrize("T_target", [1, 127, 129, 300, 1025])
def test_token_count_sweep_mxfp8(H, Q, T_target):
    m = W.TINY
    blob = H.cached_blob(m, 1)
    rng = np.random.default_rng(T_target)
    tl, left = [], T_target
    while left > 0:
        s = int(min(left, rng.integers(1, 256)))
        tl.append(s - 1)
        left -= s
    T = len(tl) + sum(tl)
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    ref = Q.encode_mxfp8(blob, W.blob_layout(m), m, emb, tl, 1, 1)
    g = H.GpuTE(m, len(tl), T, blob, weight_dtype=1)
    _assert_mx(PM.stack_metrics(g.encode(emb, tl, 1, 1), ref, emb), f"mxfp8 T={T}")
    g.close()


_W28 = {}     # quantised 28-layer weights of the oracle, shared by the three workloads below (same blob: seed 1)


@pytest.mark.timeout(1500)
@pytest.mark.parametrize("cfg_id,frames", [(3, [0, 3]), (4, [0, 15]), (5, [8])])
def test_28_layer_stacks_mxfp8_sampled_frames(H, Q, cfg_id, frames):
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    g = H.GpuTE(m, w.n_frames, T, blob, weight_dtype=1)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    assert np.isfinite(out).all()
    ref = Q.encode_mxfp8(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, frames=frames, weights_cache=_W28)
    met = PM.stack_metrics(out, ref, emb, ch)
    print(f"cfg{cfg_id} mxfp8: {met}")
    _assert_mx(met, f"cfg{cfg_id} mxfp8", deep=True)
    g.close()


@pytest.mark.timeout(900)
@pytest.mark.parametrize("cfg_id,layer", [(4, 13), (4, 27), (5, 6), (3, 20)])
def test_one_layer_every_row_full_size_mxfp8(H, Q, cfg_id, layer):
    """Teacher-forced ONE layer at depth, over ALL rows at full size (cfg 4: 12 row-pair blocks x every tile of the four
    block-scaled GEMMs; cfg 5 ragged; cfg 3 the small-batch shape): the input residual is the same on both sides, so the
    shallow gates apply at any depth — this is what certifies the deep stack layer by layer."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    x_in = (emb * np.float32(1.0 + 0.05 * layer)).astype(np.float32)     # a residual-like input (outlier channels kept)
    taps = {}
    ref = Q.encode_mxfp8(blob, W.blob_layout(m), m, x_in, tl, w.grid_h, w.grid_w, layer_begin=layer, layer_end=layer + 1,
                         taps=taps)
    g = H.GpuTE(m, w.n_frames, T, blob, weight_dtype=1)
    out = g.encode(x_in, tl, w.grid_h, w.grid_w, layer_range=(layer, layer + 1))
    gt = g.taps_mx(T)
    for key in ("q", "k", "v"):
        assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_REL_L2, (cfg_id, key)
        assert PM.max_row_rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_ROW_REL_L2, (cfg_id, key)
    for key in ("attn", "act"):
        assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_MX_TAP_REL_L2, (cfg_id, key)
    e64 = x_in.astype(np.float64)
    rows = PM.row_rel_l2(out - e64, ref - e64)
    print(f"cfg{cfg_id} layer {layer} mxfp8: update {PM.rel_l2(out - e64, ref - e64):.3e}, max row {rows.max():.3e}")
    assert PM.rel_l2(out - e64, ref - e64) <= PM.GATE_MX_UPDATE_REL_L2
    assert rows.max() <= PM.GATE_MX_ROW_UPDATE_REL_L2, (int(rows.argmax()), float(rows.max()))
    g.close()


def test_identical_frames_cover_every_row_mxfp8(H, Q):
    """cfg 4 at full size, full depth: identical frames must come out bitwise identical (every row block, every tile)."""
    w, blob, tl, T, emb, ch = H.workload_inputs(4)
    m = w.model
    S = T // w.n_frames
    same = np.concatenate([emb[:S]] * w.n_frames)
    g = H.GpuTE(m, w.n_frames, T, blob, weight_dtype=1)
    out = g.encode(same, tl, w.grid_h, w.grid_w)
    for b in range(1, w.n_frames):
        assert np.array_equal(out[b * S:(b + 1) * S], out[:S]), b
    g.close()


def test_mxfp8_create_refuses_what_it_cannot_run(H):
    import paper_2606_05981_b200 as te
    m = W.TEModelConfig(n_layers=1, hidden=256, n_q_heads=6, n_kv_heads=2, head_dim=64, ffn=512, rope_sections=(8, 12, 12))
    h = te.c_void_p()
    cfg = te.make_config(m, 2, 128, weight_dtype=1)                    # G = 3: no quantising attention epilogue
    assert te.lib().te_create(te.byref(cfg), 0, te.byref(h)) == te.TE_ERR_UNSUPPORTED
    cfg = te.make_config(W.TINY, 2, 128, max_prefix_tokens=16, weight_dtype=1)
    assert te.lib().te_create(te.byref(cfg), 0, te.byref(h)) == te.TE_ERR_UNSUPPORTED
