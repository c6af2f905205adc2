"""Pins for the oracle's block-scaled (MX) e4m3 quantisation (block-scaled variant): the exponent of
every block of 32 against its definition by brute force, the codes against the e4m3 pins of test_oracle_fp8_pins.py,
invariants.  -m "not gpu"."""
import numpy as np
import torch

from oracle import sq_oracle as O


def test_block_exponent_is_the_smallest_that_avoids_saturation():
    gen = torch.Generator().manual_seed(3)
    X = (torch.randn(40, 200, generator=gen) * torch.exp(torch.rand(40, 1, generator=gen) * 12 - 8)).to(torch.bfloat16)
    X[5] = 0
    X[6, :32] = 448.0; X[7, :32] = 900.0; X[8, :32] = 0.4375          # exactly 448 * 2^0, just above 448 * 2^1 (900 is a bf16 value), 448 * 2^-10
    codes, e = O.quantize_mx(X)
    assert codes.shape == (40, 200) and e.shape == (40, 7) and e.dtype == np.int32      # 200 = 6 * 32 + 8: ragged last block
    x = X.double().numpy()
    for r in range(40):
        for b in range(7):
            blk = np.abs(x[r, 32 * b:32 * b + 32])
            amax = blk.max()
            if amax == 0:
                assert e[r, b] == -127 and not codes[r, 32 * b:32 * b + 32].any()
                continue
            # brute force over every exponent: the smallest e with amax <= 448 * 2^e
            want = min(k for k in range(-140, 140) if amax <= 448.0 * 2.0 ** k)
            assert e[r, b] == want, (r, b, amax, e[r, b], want)
    assert e[6, 0] == 0 and e[7, 0] == 2 and e[8, 0] == -10


def test_codes_are_the_nearest_e4m3_of_the_exactly_scaled_values():
    gen = torch.Generator().manual_seed(4)
    X = (torch.randn(16, 96, generator=gen) * 0.02).to(torch.bfloat16)
    codes, e = O.quantize_mx(X)
    y = X.double().numpy() / np.repeat(2.0 ** e.astype(np.float64), 32, axis=1)
    assert np.abs(y).max() <= 448.0                                    # nothing saturates
    assert np.abs(y).reshape(16, 3, 32).max(axis=2).min() > 224.0      # and the scale is tight: the block maximum uses the top binade
    np.testing.assert_array_equal(codes, O.round_to_e4m3(y))
    deq = O.dequantize_mx(codes, e).numpy()
    x = X.double().numpy()
    blk_scale = np.repeat(2.0 ** e.astype(np.float64), 32, axis=1)
    assert np.all(np.abs(deq - x) <= np.maximum(2.0 ** -4 * np.abs(x), 2.0 ** -10 * blk_scale) * (1 + 1e-12))
    # per-block scaling beats one scale per row: an outlier only costs its own block
    X2 = X.clone(); X2[:, 0] = 8.0
    c2, e2 = O.quantize_mx(X2)
    np.testing.assert_array_equal(c2[:, 32:], codes[:, 32:])
    np.testing.assert_array_equal(e2[:, 1:], e[:, 1:])


def test_power_of_two_rescaling_moves_the_exponents_only():
    gen = torch.Generator().manual_seed(5)
    X = torch.randn(8, 64, generator=gen).to(torch.bfloat16)
    c1, e1 = O.quantize_mx(X)
    c2, e2 = O.quantize_mx((X.float() * 16).to(torch.bfloat16))
    np.testing.assert_array_equal(c1, c2)
    np.testing.assert_array_equal(e2, e1 + 4)
    np.testing.assert_array_equal(O.dequantize_mx(c2, e2).numpy(), 16 * O.dequantize_mx(c1, e1).numpy())
