"""`-m gpu` parity tests of the MXFP4-weight variant (te_config.weight_dtype = 2: FP4 E2M1 weights x MXFP8 activations on
tcgen05.mma.kind::mxf8f6f4; reading Q32 of DESIGN.md §3) against oracle/te_mxfp8.py (encode_mxfp8(fp4_weights=True)).
Integer work (codes, scales) bit-exact; the mixed-format GEMM alone to fp32-accumulation accuracy; stacks within the
gates of the MXFP8 variant (the weights are bit-identical on both sides, the activations are quantised as there)."""
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
def H():
    import gpu_helpers
    return gpu_helpers


def _weights_like(rng, rows, K):
    x = (rng.standard_normal((rows, K)) * np.exp(rng.uniform(-4, 2, size=(rows, 1)))).astype(np.float32)
    if rows >= 8:
        x[::5, 32:64] = 0.0                    # all-zero blocks
        x[2, 70] = 6.0 * 2.0 ** 3              # exactly on the 1.5 * 2^n boundary of the scale rule
        x[3, 100:108] = [0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0, 6.0]      # the grid's midpoints (if the block's X is 1)
        x[3, 96] = 6.0
    return W.f32_to_bf16_bits(x)


@pytest.mark.parametrize("rows,K", [(128, 128), (300, 512), (2048, 6144)])
def test_fp4_quantiser_bit_exact(H, Q, rows, K):
    import torch
    import paper_2606_05981_b200 as te
    bits = _weights_like(np.random.default_rng(rows + K), rows, K)
    src = torch.from_numpy(bits.view(np.int16)).cuda()
    codes = torch.zeros((rows, K // 2), dtype=torch.uint8, device="cuda")
    sft = torch.full(((rows + 127) // 128, K // 128, 512), 0xEE, dtype=torch.uint8, device="cuda")
    te.te_debug_mx_quantise_fp4(0, src, rows, K, codes, sft)
    want_codes, want_sf = Q.quantise_fp4(H.bf16_bits_to_f64(bits).reshape(rows, K))
    assert np.array_equal(H.untile_scales(sft.cpu().numpy(), rows, K), want_sf)
    got = codes.cpu().numpy()
    lo, hi = got & 0xF, got >> 4
    got_codes = np.empty((rows, K), dtype=np.uint8)
    got_codes[:, 0::2], got_codes[:, 1::2] = lo, hi                      # element 2i in the low nibble
    same = (got_codes == want_codes) | (((got_codes | want_codes) & 0x7) == 0)   # +0 and -0 are the same value
    assert same.all(), np.argwhere(~same)[:5]


@pytest.mark.parametrize("M,N,K,bn", [(128, 128, 128, 128), (256, 256, 128, 256), (1, 128, 256, 128), (300, 512, 256, 256),
                                       (517, 768, 896, 128), (3072, 4096, 2048, 128), (3072, 2048, 6144, 256)])
def test_gemm_fp8_x_fp4_vs_fp64_of_the_dequantised_operands(H, Q, M, N, K, bn):
    """E4M3 x E2M1 block-scaled main loop alone: A quantised to MXFP8, B to MXFP4 (packed nibbles, unpacked into the
    128-byte swizzled rows by the tensor map) on the device; the product must equal the fp64 product of the dequantised
    operands to fp32-accumulation accuracy.  A wrong nibble order, element format or scale byte is an O(1) error."""
    import torch
    import paper_2606_05981_b200 as te
    rng = np.random.default_rng(M + 3 * N + K)
    a = W.f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    b = _weights_like(rng, N, K)
    A = Q.fake_quant(H.bf16_bits_to_f64(a).reshape(M, K))
    B = Q.fake_quant_fp4(H.bf16_bits_to_f64(b).reshape(N, K))
    ref = A @ B.T
    c = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    te.te_debug_gemm_mxfp4(0, torch.from_numpy(a.view(np.int16)).cuda(), torch.from_numpy(b.view(np.int16)).cuda(), c,
                           M, N, K, bn)
    out = c.cpu().numpy()
    assert np.isfinite(out).all()
    assert PM.rel_l2(out, ref) < 1e-5
    scale = np.linalg.norm(A, axis=1)[:, None] * np.maximum(np.linalg.norm(B, axis=1)[None, :], 1e-30)
    assert np.max(np.abs(out - ref) / scale) < 1e-5


def test_cfg1_stack_mxfp4(H, Q):
    from oracle import te_oracle as O
    w, blob, tl, T, emb, ch = H.workload_inputs(1)
    lay = W.blob_layout(w.model)
    ref = Q.encode_mxfp8(blob, lay, w.model, emb, tl, 4, 4, fp4_weights=True)
    g = H.GpuTE(w.model, w.n_frames, T, blob, weight_dtype=2)
    out = g.encode(emb, tl, 4, 4)
    met = PM.stack_metrics(out, ref, emb)
    print("cfg1 mxfp4:", met)
    assert PM.passes_mx_gates(met), met
    assert np.array_equal(out, g.encode(emb, tl, 4, 4, use_graph=0))
    # a different network from both the MXFP8 one and the unquantised one
    ref8 = Q.encode_mxfp8(blob, lay, w.model, emb, tl, 4, 4)
    plain = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    e = PM.rel_l2(out - emb, ref - emb)
    assert PM.rel_l2(out - emb, ref8 - emb) > 2 * e and PM.rel_l2(out - emb, plain - emb) > 2 * e
    g.close()


def test_layer0_taps_mxfp4(H, Q):
    w, blob, tl, T, emb, ch = H.workload_inputs(2)
    m = w.model
    taps = {}
    ref = Q.encode_mxfp8(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, layer_begin=0, layer_end=1, taps=taps,
                         fp4_weights=True)
    g = H.GpuTE(m, w.n_frames, T, blob, weight_dtype=2)
    out = g.encode(emb, tl, w.grid_h, w.grid_w, layer_range=(0, 1))
    gt = g.taps_mx(T)
    for key in ("q", "k", "v"):
        assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_TAP_REL_L2, (key, PM.rel_l2(gt[key], taps[key][0]))
    for key in ("attn", "act"):
        assert PM.rel_l2(gt[key], taps[key][0]) <= PM.GATE_MX_TAP_REL_L2, (key, PM.rel_l2(gt[key], taps[key][0]))
    e64 = emb.astype(np.float64)
    assert PM.rel_l2(out - e64, ref - e64) <= PM.GATE_MX_UPDATE_REL_L2
    assert PM.max_row_rel_l2(out - e64, ref - e64) <= PM.GATE_MX_ROW_UPDATE_REL_L2
    g.close()


@pytest.mark.timeout(900)
@pytest.mark.parametrize("cfg_id,layer", [(4, 13), (3, 20), (5, 6)])
def test_one_layer_every_row_full_size_mxfp4(H, Q, cfg_id, layer):
    """Teacher-forced ONE layer at depth over ALL rows at full size, as for the MXFP8 variant."""
    w, blob, tl, T, emb, ch = H.workload_inputs(cfg_id)
    m = w.model
    x_in = (emb * np.float32(1.0 + 0.05 * layer)).astype(np.float32)
    ref = Q.encode_mxfp8(blob, W.blob_layout(m), m, x_in, tl, w.grid_h, w.grid_w, layer_begin=layer, layer_end=layer + 1,
                         fp4_weights=True)
    g = H.GpuTE(m, w.n_frames, T, blob, weight_dtype=2)
    out = g.encode(x_in, tl, w.grid_h, w.grid_w, layer_range=(layer, layer + 1))
    e64 = x_in.astype(np.float64)
    rows = PM.row_rel_l2(out - e64, ref - e64)
    print(f"cfg{cfg_id} layer {layer} mxfp4: update {PM.rel_l2(out - e64, ref - e64):.3e}, max row {rows.max():.3e}")
    assert PM.rel_l2(out - e64, ref - e64) <= PM.GATE_MX_UPDATE_REL_L2
    assert rows.max() <= PM.GATE_MX_ROW_UPDATE_REL_L2, (int(rows.argmax()), float(rows.max()))
    g.close()


@pytest.mark.timeout(1500)
def test_28_layer_stack_mxfp4_sampled_frames(H, Q):
    w, blob, tl, T, emb, ch = H.workload_inputs(4)
    m = w.model
    g = H.GpuTE(m, w.n_frames, T, blob, weight_dtype=2)
    out = g.encode(emb, tl, w.grid_h, w.grid_w)
    assert np.isfinite(out).all()
    S = T // w.n_frames
    ref = Q.encode_mxfp8(blob, W.blob_layout(m), m, emb, tl, w.grid_h, w.grid_w, frames=[0, 15], fp4_weights=True)
    met = PM.stack_metrics(out, ref, emb, ch)
    print(f"cfg4 mxfp4: {met}")
    assert PM.passes_mx_gates(met, deep=True), met
    g.close()
