"""Pins of the MXFP8 quantiser (oracle/te_mxfp8.py, readings Q24-Q27 of DESIGN.md §3)
against what the formats fix: hand-worked E4M3 values and rounding cases, the E8M0 scale rule on worked amax
values, invariants of the block format, and the quantised network's special cases.  CPU only."""
import numpy as np
import pytest

import workloads as W
from oracle import te_mxfp8 as Q
from oracle import te_oracle as O


def test_e4m3_decode_hand_worked_codes():
    """E4M3 'fn' values typed from the format definition (bias 7, 3 mantissa bits, no inf, max 448)."""
    want = {0x00: 0.0, 0x01: 2.0 ** -9, 0x07: 7 * 2.0 ** -9, 0x08: 2.0 ** -6, 0x09: 1.125 * 2.0 ** -6,
            0x38: 1.0, 0x39: 1.125, 0x3C: 1.5, 0x40: 2.0, 0x47: 3.75, 0x77: 240.0, 0x78: 256.0, 0x7E: 448.0,
            0xB8: -1.0, 0xFE: -448.0, 0x81: -(2.0 ** -9)}
    for code, val in want.items():
        assert Q.e4m3_decode(np.uint8(code)) == val, hex(code)
    assert np.isnan(Q.e4m3_decode(np.uint8(0x7F)))
    v = Q.e4m3_decode(np.arange(0x7F, dtype=np.uint8))
    assert np.all(np.diff(v) > 0)                                  # codes 0x00..0x7E are strictly increasing


def test_e4m3_encode_round_to_nearest_even_hand_worked():
    """Rounding cases worked by hand: between 1.0 (0x38, even) and 1.125 (0x39, odd) the midpoint 1.0625 goes to
    the even code; between 1.125 and 1.25 (0x3A) the midpoint 1.1875 goes up to 0x3A; the subnormal step is 2^-9."""
    cases = [(1.0, 0x38), (1.0624, 0x38), (1.0625, 0x38), (1.0626, 0x39), (1.1875, 0x3A), (1.18, 0x39),
             (448.0, 0x7E), (440.0, 0x7E), (432.0, 0x7E), (431.9, 0x7D), (416.0, 0x7D), (400.0, 0x7C), (0.0, 0x00),
             (2.0 ** -10, 0x00), (2.0 ** -10 * 1.01, 0x01), (3 * 2.0 ** -10, 0x02), (2.0 ** -6, 0x08),
             (-1.0625, 0xB8), (-3.9, 0xC8), (247.9, 0x77), (248.0, 0x78), (15.5 * 2.0 ** -10, 0x08)]
    for v, code in cases:
        assert Q.e4m3_encode_rne(np.float64(v)) == code, (v, hex(code), hex(int(Q.e4m3_encode_rne(np.float64(v)))))
    codes = np.arange(0x7F, dtype=np.uint8)
    assert np.array_equal(Q.e4m3_encode_rne(Q.e4m3_decode(codes)), codes)          # every value is a fixed point
    assert np.array_equal(Q.e4m3_encode_rne(-Q.e4m3_decode(codes[1:])), codes[1:] | 0x80)


def test_value_rounding_equals_code_rounding():
    """e4m3_round (rint on the binade's step) == decode(encode) (nearest-value table search, ties to the even code)
    on every midpoint, every grid value and a dense random sample; fake_quant == dequantise(quantise)."""
    grid = Q.e4m3_decode(np.arange(0x7F, dtype=np.uint8))
    mids = (grid[1:] + grid[:-1]) / 2
    rng = np.random.default_rng(3)
    v = np.concatenate([grid, mids, np.nextafter(mids, 0), np.nextafter(mids, 1e9), rng.uniform(0, 448, 200000),
                        np.exp(rng.uniform(np.log(2.0 ** -12), np.log(448.0), 200000))])
    v = np.concatenate([v, -v])
    assert np.array_equal(Q.e4m3_round(v), Q.e4m3_decode(Q.e4m3_encode_rne(v)))
    x = (rng.standard_normal((50, 512)) * np.exp(rng.uniform(-30, 30, size=(50, 1)))).astype(np.float32)
    x[:, 7] *= 1000
    assert np.array_equal(Q.fake_quant(x), Q.dequantise(*Q.quantise(x)))


def test_scale_code_hand_worked_amax():
    """Q25: the smallest power of two X with amax / X <= 448.  448 = 1.75 * 2^8."""
    cases = [(448.0, 127), (448.0001, 128), (449.0, 128), (896.0, 128), (897.0, 129), (1.0, 127 - 8),
             (1.75, 127 - 8), (1.7500001, 127 - 7), (224.0, 126), (225.0, 127), (3000.0, 130), (1160.0, 129),
             (0.0, 0), (37.0, 124), (2.0 ** -20, 127 - 28)]
    for amax, code in cases:
        got = int(Q.scale_code(np.float32(amax)))
        assert got == code, (amax, code, got)
        if amax > 0:
            X = 2.0 ** (got - 127)
            assert np.float32(amax) / X <= 448.0 and np.float32(amax) / (X / 2) > 448.0


def test_quantise_worked_block_with_an_outlier():
    """One block holding a x1000-class outlier (max 1160): amax = 1160 -> X = 4 (code 129); the
    small values land on the subnormal grid of step 4 * 2^-9, hand-computed."""
    x = np.zeros(32, dtype=np.float32)
    x[0], x[1], x[2], x[3], x[4] = 1160.0, -854.0, 1.0, 0.01, 0.0039
    codes, sc = Q.quantise(x)
    assert sc.shape == (1,) and sc[0] == 129
    dq = Q.dequantise(codes, sc)
    assert dq[0] == 1152.0            # 290 -> nearest of (288, 320) = 288 -> * 4
    assert dq[1] == -832.0            # 213.5 -> grid (208, 224) -> 208 -> * 4
    assert dq[2] == 1.0               # 0.25 is exact
    assert dq[3] == 0.0078125         # 0.0025 -> subnormal grid step 2^-9: 1.28 steps -> 1 step = 2^-9 -> * 4
    assert dq[4] == 0.0               # 0.000975 = 0.499 steps -> 0
    assert np.all(dq[5:] == 0.0)


def test_quantiser_invariants():
    rng = np.random.default_rng(0)
    x = (rng.standard_normal((64, 256)) * np.exp(rng.uniform(-20, 20, size=(64, 1)))).astype(np.float32)
    codes, sc = Q.quantise(x)
    assert codes.shape == x.shape and sc.shape == (64, 8)
    dq = Q.dequantise(codes, sc)
    blk = np.abs(x.astype(np.float64)).reshape(64, 8, 32)
    X = 2.0 ** (sc.astype(np.float64) - 127)
    assert np.all(blk.max(-1) / X <= 448.0) and np.all(blk.max(-1) / X > 224.0)      # never saturates, tight scale
    assert (codes & 0x7F).max() <= 0x7E                                              # no NaN code
    err = np.abs(dq - x).reshape(64, 8, 32)
    # half an ulp of the value's binade (3 mantissa bits), or half a subnormal step of the block
    bound = np.maximum(blk * 2.0 ** -4, X[..., None] * 2.0 ** -10)
    assert np.all(err <= bound * (1 + 1e-12))
    # blocks are independent; scaling a block by a power of two scales its dequantised values exactly
    y = x.copy()
    y[:, 32:64] *= np.float32(8.0)
    dq2 = Q.dequantise(*Q.quantise(y))
    assert np.array_equal(dq2[:, :32], dq[:, :32]) and np.array_equal(dq2[:, 64:], dq[:, 64:])
    assert np.array_equal(dq2[:, 32:64], dq[:, 32:64] * 8.0)
    # idempotent: quantised values are fixed points
    assert np.array_equal(Q.fake_quant(dq), dq)
    # decisions are taken on float32 values (Q27): a float64 input that rounds to the same float32 gives the same codes
    assert np.array_equal(Q.quantise(x.astype(np.float64) * (1 + 1e-12))[0], codes)


def test_quantised_network_special_cases():
    """(i) weights and activations that are exactly representable pass through the quantiser unchanged, so the MXFP8
    network equals the plain oracle there; (ii) zero projections pass the residual through exactly; (iii) frames stay
    independent; (iv) on seeded cfg-1 inputs the quantised network differs from the unquantised one by the size of
    8-bit noise, not more."""
    m = W.TINY.with_layers(1)
    lay = W.blob_layout(m)
    blob = W.make_weight_blob(m, 1)
    tl, gh, gw = [9, 4], 2, 2
    T = 2 * 4 + sum(tl)
    emb = np.random.default_rng(1).standard_normal((T, m.hidden)).astype(np.float32)
    ref = O.encode(blob, lay, m, emb, tl, gh, gw)
    out = Q.encode_mxfp8(blob, lay, m, emb, tl, gh, gw)
    upd = np.linalg.norm((out - emb) - (ref - emb)) / np.linalg.norm(ref - emb)
    assert 5e-3 < upd < 1.2e-1, upd                                  # 8-bit noise: visible, bounded
    # (ii) zero projections
    z = blob.copy()
    for name in ("Wo", "Wdown"):
        off, shape = lay[(0, name)]
        z[off:off + int(np.prod(shape))] = 0
    assert np.array_equal(Q.encode_mxfp8(z, lay, m, emb, tl, gh, gw), emb.astype(np.float64))
    # (iii) frame independence
    solo = Q.encode_mxfp8(blob, lay, m, emb[13:], tl[1:], gh, gw)
    assert np.array_equal(out[13:], solo)
    # (i) weights on the e4m3 grid (power-of-two scale 2^-6 keeps the stack tame) are fixed points of the quantiser
    Wl = O.unpack_layer(blob, lay, 0)
    snapped = Q.fake_quant(Wl["Wq"])
    assert np.array_equal(Q.fake_quant(snapped), snapped)
    assert np.max(np.abs(snapped - Wl["Wq"]) / np.abs(Wl["Wq"]).max()) < 2.0 ** -4


# ---------------------------------------------------------------- MXFP4 weights (reading Q32)
def test_e2m1_codes_hand_typed():
    """All sixteen E2M1 codes from the format definition (sign, 2-bit exponent with bias 1, 1 mantissa bit)."""
    want = [0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0]
    assert Q.e2m1_decode(np.arange(8)).tolist() == want
    assert Q.e2m1_decode(np.arange(8, 16)).tolist() == [-x for x in want]


def test_e2m1_rounding_hand_worked():
    """Nearest value, ties to the even code: every midpoint of the grid typed by hand, plus off-midpoint and clamped cases."""
    v = np.asarray([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0])           # the seven midpoints
    assert Q.e2m1_encode_rne(v).tolist() == [0, 2, 2, 4, 4, 6, 6]      # -> 0, 1, 1, 2, 2, 4, 4
    assert Q.e2m1_encode_rne(-v).tolist() == [8, 10, 10, 12, 12, 14, 14]
    v2 = np.asarray([0.2, 0.3, 0.74, 0.76, 2.49, 2.51, 4.99, 5.01, 6.0, 7.5, 100.0])
    assert Q.e2m1_encode_rne(v2).tolist() == [0, 1, 1, 2, 4, 5, 6, 7, 7, 7, 7]
    # decode(encode) is the identity on the grid and idempotent everywhere
    g = Q.e2m1_decode(np.arange(16))
    assert np.array_equal(Q.e2m1_decode(Q.e2m1_encode_rne(g))[1:], g[1:])
    x = np.random.default_rng(0).uniform(-6, 6, 1000)
    once = Q.e2m1_decode(Q.e2m1_encode_rne(x))
    assert np.array_equal(Q.e2m1_decode(Q.e2m1_encode_rne(once)), once)
    assert np.max(np.abs(once - x)) <= 1.0                              # half of the widest grid step (4 -> 6)


def test_e2m1_round_equals_decode_of_encode():
    """The value-domain rounding used by fake_quant_fp4 is the table-search quantiser: on every midpoint, every grid
    value, both signs, a dense sweep, and beyond the clamp."""
    pts = np.concatenate([[0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0], Q._GRID4, np.linspace(0, 7.5, 6001),
                          np.nextafter([0.25, 0.75, 1.25, 1.75, 2.0, 2.5, 3.5, 4.0, 5.0], 0),
                          np.nextafter([0.25, 0.75, 1.25, 1.75, 2.0, 2.5, 3.5, 4.0, 5.0], 10)])
    pts = np.concatenate([pts, -pts])
    assert np.array_equal(Q.e2m1_round(pts), Q.e2m1_decode(Q.e2m1_encode_rne(pts)))
    x = np.random.default_rng(1).standard_normal((64, 256)).astype(np.float32) * 3
    c, s = Q.quantise_fp4(x)
    assert np.array_equal(Q.fake_quant_fp4(x), Q.dequantise_fp4(c, s))


def test_fp4_scale_codes_worked():
    """Smallest power of two X with amax / X <= 6 (= 1.5 * 2^2): worked from the float32 fields."""
    amax = np.asarray([6.0, 6.0001, 1.0, 1.5, 1.51, 0.0, 12.0, 0.02, 3.0e-3], dtype=np.float32)
    code = Q.scale_code_fp4(amax)
    assert code.tolist()[:7] == [127, 128, 125, 125, 126, 0, 128]
    X = 2.0 ** (code.astype(np.float64) - 127)
    nz = amax > 0
    assert np.all(amax[nz] / X[nz] <= 6.0) and np.all(amax[nz] / (X[nz] / 2) > 6.0)       # smallest such power of two


def test_fp4_block_worked_and_packing():
    """One block typed by hand: amax 3.0 -> X = 0.5 (3 / 0.5 = 6), elements v / 0.5 rounded to the grid."""
    blk = np.zeros(32, dtype=np.float32)
    blk[:8] = [3.0, -1.5, 0.26, 0.74, 1.1, -0.6, 2.2, 0.1]
    codes, sc = Q.quantise_fp4(blk[None, :])
    assert sc.tolist() == [[126]]
    # v / 0.5 = 6, -3, 0.52, 1.48, 2.2, -1.2, 4.4, 0.2  ->  6, -3, 0.5, 1.5, 2, -1, 4, 0
    assert codes[0, :8].tolist() == [7, 13, 1, 3, 4, 10, 6, 0]
    assert Q.dequantise_fp4(codes, sc)[0, :8].tolist() == [3.0, -1.5, 0.25, 0.75, 1.0, -0.5, 2.0, 0.0]
    packed = Q.pack_fp4(codes)
    assert packed.shape == (1, 16) and packed[0, :4].tolist() == [7 | (13 << 4), 1 | (3 << 4), 4 | (10 << 4), 6 | (0 << 4)]
    assert np.array_equal(Q.fake_quant_fp4(blk[None, :]), Q.dequantise_fp4(codes, sc))


def test_fp4_network_special_cases():
    """The W4A8 network: weights exactly representable in MXFP4 make it the MXFP8 network; quantisation noise of the
    weights is the expected ~10 % class on a GEMM (24 dB SQNR ballpark of a 1-mantissa-bit format)."""
    import workloads as W
    from oracle import te_oracle as O
    m = W.TINY
    blob = W.make_weight_blob(m, 1)
    lay = W.blob_layout(m)
    Wl = O.unpack_layer(blob, lay, 0)
    W4 = Q.quantise_layer_weights_fp4(Wl)
    again = Q.quantise_layer_weights_fp4(W4)                           # idempotent
    assert all(np.array_equal(W4[k], again[k]) for k in ("Wq", "Wo", "Wgate", "Wdown"))
    assert np.array_equal(W4["g1"], Wl["g1"])                           # gains untouched
    rel = np.linalg.norm(W4["Wq"] - Wl["Wq"]) / np.linalg.norm(Wl["Wq"])
    assert 0.05 < rel < 0.2, rel
    # MXFP4-representable weights: MXFP8 quantisation leaves them unchanged too -> the two networks coincide
    w8 = Q.quantise_layer_weights(W4)
    assert all(np.array_equal(w8[k], W4[k]) for k in ("Wq", "Wk", "Wv", "Wo", "Wgate", "Wup", "Wdown"))
