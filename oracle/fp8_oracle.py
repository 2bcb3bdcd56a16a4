"""CPU oracle for FP8 (e4m3) cold-pool pages (NEXT-4, "FP8 KV pages": the host-link half, S5).

TEST INFRASTRUCTURE - NOT PRODUCT CODE (same rules as oracle/lsa_oracle.py).

What is computed (R34-R36; SURVEY.md 8(f) NEXT-4 "FP8 KV pages"; the paper itself only says that
non-recalled CSA KV lives in a CPU cold mirror and is recalled page by page over the host link):
  * a cold page holds its K block and its V block as e4m3 codes (1 sign, 4 exponent bits with bias 7, 3 mantissa
    bits; no infinities; S.1111.111 is NaN; largest finite value 448 - the "fn" variant every GPU library uses)
    plus one fp32 scale per block;
  * RECALL (S5) dequantises while it copies: hot value = bf16_rne(fp32(code) * scale).  With a power-of-two
    scale this is exact (a code has 4 significant bits, bf16 has 8);
  * EXPORT quantises a bf16 block: e = floor(log2(max |x|)) - 7 taken from the exponent field of the largest
    magnitude (so max |x| * 2^-e lies in [128, 256) <= 448), scale = 2^e, code = e4m3_rne(x * 2^-e) with
    round-to-nearest-even in the e4m3 grid (the product is exact in fp32).  An all-zero block has scale 1.

Everything is written out from the format's definition: the 256-entry value table, nearest-even rounding as a
search over the grid's midpoints.  No library cast is used here; torch's float8_e4m3fn cast is one of the PINS
(tests/test_fp8_oracle_pins.py), together with closed-form codes, hand-checked ties and round-trip bounds.
"""
from __future__ import annotations

from typing import Tuple

import numpy as np

E4M3_MAX = 448.0


def e4m3_table() -> np.ndarray:
    """float64[256]: the value of every code.  code = s eeee mmm; e = 0: subnormal m/8 * 2^-6; else (1 + m/8) * 2^(e-7);
    e = 15, m = 7 is NaN (there are no infinities)."""
    t = np.empty(256, dtype=np.float64)
    for code in range(256):
        s, e, m = code >> 7, (code >> 3) & 15, code & 7
        if e == 15 and m == 7:
            v = np.nan
        elif e == 0:
            v = (m / 8.0) * 2.0 ** -6
        else:
            v = (1.0 + m / 8.0) * 2.0 ** (e - 7)
        t[code] = -v if s else v
    return t


_TABLE = e4m3_table()
_POS = _TABLE[:127]                       # codes 0x00..0x7E: 0 .. 448, strictly increasing
_MID = (_POS[:-1] + _POS[1:]) / 2.0       # midpoint between code i and code i + 1


def e4m3_decode(codes: np.ndarray) -> np.ndarray:
    """uint8 codes -> float64 values (NaN for 0x7F / 0xFF)."""
    return _TABLE[np.asarray(codes, dtype=np.uint8)]


def e4m3_encode_rne(x: np.ndarray) -> np.ndarray:
    """float array -> uint8 codes: nearest grid value, ties to the code with an even mantissa (even code), magnitudes
    above 448 saturate to 448 (the grid has no infinity).  -0.0 and negative values that round to zero keep their sign
    bit, like the hardware conversion.  Inputs must not be NaN."""
    x = np.asarray(x, dtype=np.float64)
    a = np.abs(x)
    i = np.searchsorted(_MID, a, side="left")            # a <= MID[i]  ->  candidate code i (a > every midpoint: 126)
    i = np.minimum(i, 126)
    tie = (i < 126) & (a == _MID[np.minimum(i, 125)])    # exactly half way between code i and code i + 1
    i = np.where(tie & (i % 2 == 1), i + 1, i)           # ties go to the even code
    return (i | (np.signbit(x).astype(np.int64) << 7)).astype(np.uint8)


def bf16_rne_bits(x: np.ndarray) -> np.ndarray:
    """float32 array -> bfloat16 bit patterns (uint16), round to nearest even (finite inputs)."""
    u = np.asarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    r = u + 0x7FFF + ((u >> 16) & 1)
    return (r >> 16).astype(np.uint16)


def dequant_block(codes: np.ndarray, scale: float) -> np.ndarray:
    """RECALL of one block: bf16 bits of fp32(code) * scale, the product taken in fp32 and rounded once (RNE)."""
    v = e4m3_decode(codes).astype(np.float32) * np.float32(scale)
    return bf16_rne_bits(v)


def dequant_page(codes: np.ndarray, scales) -> np.ndarray:
    """codes uint8 [2][C][D], scales (scale_K, scale_V) -> hot page image, bf16 bits [2][C][D]."""
    return np.stack([dequant_block(codes[0], scales[0]), dequant_block(codes[1], scales[1])])


def block_exponent(x_f32: np.ndarray) -> int:
    """e such that max |x| * 2^-e is in [128, 256): the unbiased exponent of the largest magnitude minus 7, read from the
    exponent FIELD of its fp32 pattern (no logarithm).  Zero / subnormal-only blocks: 0 (scale 1).  Clamped to [-120, 120]."""
    m = np.max(np.abs(np.asarray(x_f32, dtype=np.float32)))
    field = int(np.float32(m).view(np.uint32) >> 23) & 0xFF
    if field == 0:
        return 0
    return max(-120, min(120, field - 127 - 7))


def quantize_block(x_f32: np.ndarray) -> Tuple[np.ndarray, float]:
    """EXPORT of one block (float32 values, e.g. widened bf16): (uint8 codes, fp32 scale = 2^e)."""
    e = block_exponent(x_f32)
    scaled = np.asarray(x_f32, dtype=np.float32).astype(np.float64) * 2.0 ** (-e)      # exact: a power of two
    return e4m3_encode_rne(scaled), float(2.0 ** e)


def quantize_page(page_f32: np.ndarray):
    """page [2][C][D] float32 -> (codes uint8 [2][C][D], (scale_K, scale_V))."""
    ck, sk = quantize_block(page_f32[0])
    cv, sv = quantize_block(page_f32[1])
    return np.stack([ck, cv]), (sk, sv)
