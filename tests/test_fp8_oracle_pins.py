"""Pins for oracle/fp8_oracle.py (FP8 e4m3 cold pages, R34-R36).  CPU only.

The oracle writes the e4m3 grid, nearest-even rounding and the block-scale rule out from their definitions; here
they are tied to things other than themselves: closed-form codes of the format, ties worked by hand, torch's
float8_e4m3fn casts (a library routine, both directions, all 256 codes and a million random values), round-trip
error bounds of a 3-bit mantissa, and exactness of power-of-two dequantisation."""
import numpy as np
import pytest
import torch

from oracle.fp8_oracle import (E4M3_MAX, bf16_rne_bits, block_exponent, dequant_block, dequant_page, e4m3_decode,
                               e4m3_encode_rne, e4m3_table, quantize_block, quantize_page)


def test_table_closed_forms():
    t = e4m3_table()
    want = {0x00: 0.0, 0x01: 2.0 ** -9, 0x07: 7 * 2.0 ** -9, 0x08: 2.0 ** -6, 0x09: 1.125 * 2.0 ** -6, 0x38: 1.0, 0x3C: 1.5,
            0x40: 2.0, 0x70: 128.0, 0x77: 240.0, 0x78: 256.0, 0x7E: 448.0, 0xB8: -1.0, 0xFE: -448.0}
    for code, v in want.items():
        assert t[code] == v, hex(code)
    assert np.isnan(t[0x7F]) and np.isnan(t[0xFF]) and np.signbit(t[0x80]) and t[0x80] == 0.0
    pos = t[:0x7F]
    assert np.all(np.diff(pos) > 0) and pos[-1] == E4M3_MAX            # 127 codes, strictly increasing up to 448
    assert np.array_equal(t[0x80:0xFF], -pos)                          # sign bit mirrors the grid
    # spacing: 8 codes per binade, each binade twice as wide as the one below (3 mantissa bits)
    for e in range(1, 15):
        seg = pos[8 * e: 8 * e + 8] if e < 15 else pos[8 * e:]
        assert np.allclose(np.diff(seg), 2.0 ** (e - 7) / 8.0, rtol=0, atol=0)


def test_decode_and_encode_agree_with_the_library_cast():
    codes = np.arange(256, dtype=np.uint8)
    lib = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float32).numpy().astype(np.float64)
    mine = e4m3_decode(codes)
    assert np.array_equal(np.isnan(lib), np.isnan(mine))
    ok = ~np.isnan(lib)
    assert np.array_equal(lib[ok], mine[ok]) and np.array_equal(np.signbit(lib[ok]), np.signbit(mine[ok]))
    g = np.random.default_rng(11)
    x = np.concatenate([g.uniform(-448, 448, 400000), g.standard_normal(400000), g.standard_normal(200000) * 2.0 ** -8,
                        mine[ok], (mine[ok][:-1] + mine[ok][1:]) / 2]).astype(np.float32)
    x = x[np.abs(x) <= 448]
    lib_codes = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    my_codes = e4m3_encode_rne(x)
    nz = e4m3_decode(my_codes) != 0                                    # (the sign of a zero result is not compared)
    assert np.array_equal(lib_codes[nz], my_codes[nz])
    assert np.all(e4m3_decode(lib_codes[~nz]) == 0)


def test_ties_and_saturation_by_hand():
    cases = [(1.0625, 0x38),          # half way 1.0 (0x38, even) .. 1.125 (0x39): even code
             (1.1875, 0x3A),          # half way 1.125 (0x39) .. 1.25 (0x3A): even code
             (1.06, 0x38), (1.07, 0x39),
             (2.0 ** -10, 0x00),      # half way 0 .. smallest subnormal 2^-9: even code 0
             (3 * 2.0 ** -10, 0x02),  # half way code 1 .. code 2
             (7.5 * 2.0 ** -9, 0x08),  # half way largest subnormal (0x07) .. smallest normal (0x08)
             (448.0, 0x7E), (460.0, 0x7E), (1000.0, 0x7E), (-1000.0, 0xFE), (-1.0625, 0xB8), (0.0, 0x00)]
    for x, code in cases:
        assert int(e4m3_encode_rne(np.array([x]))[0]) == code, (x, hex(code))


def test_block_exponent_rule():
    for mx, e in [(1.0, -7), (0.2, -10), (255.9, 0), (256.0, 1), (127.99, -1), (2.0 ** -20, -27), (3.0e4, 7)]:
        x = np.array([0.0, -mx, mx / 3], dtype=np.float32)
        assert block_exponent(x) == e, mx
        s = float(np.float32(mx)) * 2.0 ** -e
        assert 128.0 <= s < 256.0
    assert block_exponent(np.zeros(5, np.float32)) == 0
    codes, scale = quantize_block(np.zeros((4, 4), np.float32))
    assert scale == 1.0 and not codes.any()


def test_round_trip_bounds_and_identity():
    g = np.random.default_rng(5)
    x = (g.standard_normal((128, 512)) / np.sqrt(512)).astype(np.float32)
    x = torch.from_numpy(x).to(torch.bfloat16).to(torch.float32).numpy()           # a bf16 block, widened
    codes, scale = quantize_block(x)
    back = e4m3_decode(codes) * scale
    normal = np.abs(x) >= 2.0 ** -6 * scale
    assert np.all(np.abs(back - x)[normal] <= np.abs(x)[normal] * 2.0 ** -4)       # half an ulp of a 3-bit mantissa
    assert np.all(np.abs(back - x)[~normal] <= 2.0 ** -10 * scale)                 # half a subnormal step
    assert np.abs(e4m3_decode(codes)).max() >= 128                                 # the block uses the top binades
    # values already on the grid come back unchanged, scale and all
    c0 = g.integers(0, 0x7F, size=(16, 64)).astype(np.uint8) | (g.integers(0, 2, size=(16, 64)).astype(np.uint8) << 7)
    c0[0, 0] = 0x75                                                                # 208: puts the maximum in [128, 256)
    c0 = np.where((c0 & 0x7F) > 0x77, c0 & 0xF7, c0).astype(np.uint8)              # keep everything below 256
    y = (e4m3_decode(c0) * 2.0 ** -9).astype(np.float32)
    c1, s1 = quantize_block(y)
    assert s1 == 2.0 ** -9 and np.array_equal(e4m3_decode(c1), e4m3_decode(c0))


def test_dequantisation_is_exact_for_power_of_two_scales_and_rounds_once_otherwise():
    codes = np.arange(256, dtype=np.uint8)
    codes = codes[(codes & 0x7F) != 0x7F].reshape(1, -1)
    for scale in (1.0, 2.0 ** -10, 2.0 ** 5):
        bits = dequant_block(codes, scale)
        val = (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
        assert np.array_equal(val, e4m3_decode(codes) * scale)
    scale = 0.0123
    bits = dequant_block(codes, scale)
    lib = (torch.from_numpy(e4m3_decode(codes).astype(np.float32)) * torch.tensor(scale, dtype=torch.float32)).to(torch.bfloat16)
    assert np.array_equal(bits, lib.view(torch.int16).numpy().view(np.uint16))
    page = np.stack([codes.reshape(2, -1), codes.reshape(2, -1)[::-1]])
    out = dequant_page(page, (0.5, 4.0))
    assert np.array_equal(out[0], dequant_block(page[0], 0.5)) and np.array_equal(out[1], dequant_block(page[1], 4.0))


def test_bf16_rounding_against_the_library():
    g = np.random.default_rng(3)
    x = np.concatenate([g.standard_normal(100000), g.standard_normal(1000) * 1e-30, [1.00390625, 1.01171875, -1.00390625]]).astype(np.float32)
    lib = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(bf16_rne_bits(x), lib)


def test_quantize_page_blocks_are_independent():
    g = np.random.default_rng(9)
    page = np.stack([g.standard_normal((8, 16)), 100 * g.standard_normal((8, 16))]).astype(np.float32)
    codes, (sk, sv) = quantize_page(page)
    ck, sk2 = quantize_block(page[0])
    cv, sv2 = quantize_block(page[1])
    assert (sk, sv) == (sk2, sv2) and sv > sk and np.array_equal(codes[0], ck) and np.array_equal(codes[1], cv)
