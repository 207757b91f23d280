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
