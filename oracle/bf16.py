"""bf16 rounding for the oracle (test infrastructure; see oracle/__init__.py).

The paper's fidelity statement is in bf16 units: the reconstructed KV "writes into
the pool within one bf16 ULP of recompute".  The oracle computes in
fp64 and rounds ONCE, directly from fp64 to bf16, round-to-nearest-even (going
through fp32 first would round twice and can land on the other neighbour).

bf16 = 1 sign, 8 exponent, 7 stored mantissa bits: 8 significant bits, the fp32
exponent range, subnormal quantum 2^-133, largest finite (2 - 2^-7) * 2^127.
"""
import numpy as np

_BF16_MAX = (2.0 - 2.0 ** -7) * 2.0 ** 127
_MIN_QUANTUM_EXP = -133          # 2^-126 (smallest normal) * 2^-7


def bf16_rne(x):
    """Nearest bf16 value to each fp64 element (ties to even), returned as fp64."""
    x = np.asarray(x, dtype=np.float64)
    _, e = np.frexp(x)                       # x = m * 2^e with 0.5 <= |m| < 1
    # 8 significant bits => spacing 2^(e-8) inside the binade [2^(e-1), 2^e)
    qexp = np.maximum(e - 8, _MIN_QUANTUM_EXP)
    scaled = np.ldexp(x, -qexp)              # exact (power-of-two scaling)
    r = np.ldexp(np.rint(scaled), qexp)      # np.rint rounds half to even
    with np.errstate(invalid="ignore"):
        r = np.where(np.abs(r) > _BF16_MAX, np.sign(r) * np.inf, r)
    return np.where(np.isfinite(x), r, x)    # inf / nan pass through


def bf16_bits(x):
    """uint16 bit pattern of bf16_rne(x)."""
    r = bf16_rne(x).astype(np.float32)       # exact: every bf16 is an fp32
    return (r.view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def bf16_from_bits(bits):
    """fp64 value of a uint16 bf16 bit pattern."""
    b = np.asarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    with np.errstate(invalid="ignore"):      # signalling-NaN patterns
        return b.view(np.float32).astype(np.float64)


def ulp_bf16(x):
    """Spacing of bf16 at |x|: 2^(floor(log2|x|) - 7), floored at the subnormal quantum."""
    x = np.abs(np.asarray(x, dtype=np.float64))
    _, e = np.frexp(x)
    return np.ldexp(1.0, np.maximum(e - 8, _MIN_QUANTUM_EXP))
