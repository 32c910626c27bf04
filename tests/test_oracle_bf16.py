"""Pins for oracle/bf16.py: hand-worked roundings, torch's independent bf16 cast, double-rounding trap."""
import numpy as np
import torch

from oracle import bf16


def test_hand_cases_ties_to_even():
    e = 2.0 ** -7                                  # bf16 spacing in [1, 2)
    cases = {
        1.0: 1.0,
        1.0 + e / 2: 1.0,                          # tie -> even mantissa (0)
        1.0 + 3 * e / 2: 1.0 + 2 * e,              # tie -> even mantissa (2)
        1.0 + e / 2 + 2.0 ** -40: 1.0 + e,         # just above the tie
        -(1.0 + 3 * e / 2): -(1.0 + 2 * e),
        0.0: 0.0,
        3.0e39: np.inf,                            # beyond the largest finite bf16
        2.0 ** -133: 2.0 ** -133,                  # smallest subnormal is kept
        2.0 ** -135: 0.0,                          # below half of it flushes to zero
    }
    for x, want in cases.items():
        assert bf16.bf16_rne(x) == want, x


def test_single_rounding_not_via_fp32():
    # x sits 2^-30 above a bf16 tie; fp64->fp32 drops the 2^-30 and the second rounding then ties DOWN.
    x = 1.0 + 2.0 ** -8 + 2.0 ** -30
    assert bf16.bf16_rne(x) == 1.0 + 2.0 ** -7
    via_fp32 = torch.tensor(np.float32(x)).to(torch.bfloat16).item()
    assert via_fp32 == 1.0                          # the trap the oracle avoids


def test_matches_torch_cast_on_fp32_inputs():
    rng = np.random.default_rng(7)
    x = np.concatenate([rng.standard_normal(200000).astype(np.float32),
                        (rng.standard_normal(20000) * 1e-39).astype(np.float32),     # bf16 subnormals
                        (rng.standard_normal(20000) * 1e38).astype(np.float32)])
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = bf16.bf16_bits(x.astype(np.float64))
    assert np.array_equal(got, want)


def test_bits_roundtrip_all_finite_patterns():
    bits = np.arange(0, 1 << 16, dtype=np.uint32).astype(np.uint16)
    vals = bf16.bf16_from_bits(bits)
    finite = np.isfinite(vals)
    back = bf16.bf16_bits(vals[finite])
    keep = bits[finite]
    assert np.array_equal(back, keep)


def test_ulp():
    assert bf16.ulp_bf16(1.0) == 2.0 ** -7
    assert bf16.ulp_bf16(1.99) == 2.0 ** -7
    assert bf16.ulp_bf16(2.0) == 2.0 ** -6
    assert bf16.ulp_bf16(-0.75) == 2.0 ** -8
    # spacing really is the gap to the next representable value
    bits = np.array([0x3F80, 0x4000, 0x0080], dtype=np.uint16)
    v = bf16.bf16_from_bits(bits)
    nxt = bf16.bf16_from_bits(bits + np.uint16(1))
    assert np.array_equal(nxt - v, bf16.ulp_bf16(v))
