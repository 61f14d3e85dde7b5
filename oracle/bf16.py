"""bfloat16 <-> float64 for the oracle (test infrastructure; see oracle/__init__.py).

bf16 tensors are carried as numpy uint16 arrays holding the raw bits.
PAPER.md:125 fixes bfloat16 inference; reading C13: every bf16 store is
round-to-nearest-even.  The oracle rounds straight from fp64 (no fp32 stop on the
way, so there is no double rounding).
"""

import numpy as np


def to_f64(bits):
    """Widen bf16 bit patterns (uint16) to float64, exactly."""
    bits = np.asarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def from_f64(x):
    """Round float64 to bf16 bit patterns, round-to-nearest-even, directly from fp64.

    bf16 = 1 sign, 8 exponent (bias 127), 7 mantissa bits.  NaN is not expected
    (the oracle asserts); +-inf and overflow map to +-inf.
    """
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert not np.isnan(x).any(), "oracle: NaN reached a bf16 store"
    b = x.view(np.uint64)
    sign = ((b >> np.uint64(63)) & np.uint64(1)).astype(np.uint32)
    exp = ((b >> np.uint64(52)) & np.uint64(0x7FF)).astype(np.int64)
    man = b & np.uint64((1 << 52) - 1)

    # normal bf16 range: keep the top 7 mantissa bits, RNE on the low 45
    e = exp - 1023 + 127
    man7 = (man >> np.uint64(45)).astype(np.int64)
    rem = man & np.uint64((1 << 45) - 1)
    half = np.uint64(1 << 44)
    round_up = (rem > half) | ((rem == half) & ((man7 & 1) == 1))
    mag = (e << 7) + man7 + round_up.astype(np.int64)  # a mantissa carry bumps the exponent

    # results below the smallest normal (2^-126): spacing is 2^-133, rint is half-even
    sub = e <= 0
    if sub.any():
        q = np.rint(np.abs(np.where(sub, x, 0.0)) * 2.0 ** 133)
        mag = np.where(sub, q.astype(np.int64), mag)

    # overflow / inf
    mag = np.where((mag >= (255 << 7)) | (exp == 0x7FF), 255 << 7, mag)
    out = (sign << np.uint32(15)) | mag.astype(np.uint32)
    return out.astype(np.uint16)
