"""Pins for the oracle's e4m3 quantisation (SURVEY 8(f)-4, FP8 variant): the code table against the format's
definition and a library view, rounding against hand-worked ties and a library routine, quantise / dequantise
invariants.  -m "not gpu"."""
import numpy as np
import torch

from oracle import sq_oracle as O


def test_e4m3_table_hand_values_and_library_view():
    v = O.e4m3_values()
    assert v[0x00] == 0.0 and v[0x38] == 1.0 and v[0x39] == 1.125 and v[0x40] == 2.0
    assert v[0x7E] == 448.0 and np.isnan(v[0x7F]) and v[0xFE] == -448.0          # no infinities: S.1111.110 is the maximum
    assert v[0x01] == 2.0 ** -9 and v[0x07] == 7 * 2.0 ** -9 and v[0x08] == 2.0 ** -6   # subnormals, first normal
    assert np.all(np.diff(v[:127]) > 0)                                          # codes 0..126 ascend
    lib = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).double().numpy()
    assert np.array_equal(np.nan_to_num(v, nan=7e9), np.nan_to_num(lib, nan=7e9))


def test_round_to_e4m3_ties_and_special_cases():
    r = lambda x: O.e4m3_values()[O.round_to_e4m3(np.array(x, dtype=np.float64))]
    assert r([1.0625])[0] == 1.0            # halfway 1.0 (mantissa 000) / 1.125 (001): even mantissa wins
    assert r([1.1875])[0] == 1.25           # halfway 1.125 (001) / 1.25 (010)
    assert r([1.06251])[0] == 1.125 and r([1.06249])[0] == 1.0
    assert r([448.0])[0] == 448.0 and r([-448.0])[0] == -448.0 and r([440.0])[0] == 448.0 and r([431.9])[0] == 416.0
    assert r([2.0 ** -10])[0] == 0.0        # halfway 0 / 2^-9: code 0 is even
    assert r([1.5 * 2.0 ** -9])[0] == 2.0 ** -8
    assert r([0.0])[0] == 0.0
    pts = O.e4m3_values()[:127]
    assert np.array_equal(r(pts), pts) and np.array_equal(r(-pts[1:]), -pts[1:])   # idempotent on code points


def test_round_to_e4m3_matches_library_routine_and_is_nearest():
    rng = np.random.default_rng(2)
    y = np.concatenate([rng.uniform(-448, 448, 100000), rng.normal(0, 0.02, 50000), rng.normal(0, 3, 50000)]).astype(np.float32)
    y = np.clip(y, -448, 448)
    c = O.round_to_e4m3(y)
    lib = torch.from_numpy(y).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(c, lib)
    v = O.e4m3_values()[c]
    pts = O.e4m3_values()[:127]
    nearest = np.abs(np.abs(y.astype(np.float64))[:2000, None] - pts[None, :]).min(axis=1)
    assert np.allclose(np.abs(v[:2000] - y[:2000].astype(np.float64)), nearest, rtol=0, atol=0)
    order = np.argsort(y)
    assert np.all(np.diff(v[order]) >= 0)                                         # monotone


def test_quantize_scales_and_error_bound():
    gen = torch.Generator().manual_seed(8)
    X = (torch.randn(12, 64, generator=gen) * torch.exp(torch.rand(12, 1, generator=gen) * 4 - 2)).to(torch.bfloat16)
    X[3] = 0
    q, s, y = O.quantize_fp8(X, per_tensor=False)
    amax = X.double().abs().amax(dim=1).numpy()
    assert q.dtype == np.uint8 and q.shape == (12, 64) and s.shape == (12,) and y.shape == (12, 64)
    assert s[3] == 1.0 and not q[3].any()                                         # all-zero row
    np.testing.assert_array_equal(s[amax > 0], amax[amax > 0] / 448.0)            # scale = amax / 448 by definition
    np.testing.assert_allclose(y * s[:, None], X.double().numpy(), rtol=1e-15)    # y = x / scale
    v = np.abs(O.e4m3_values()[q])
    assert np.all(v.max(axis=1)[amax > 0] == 448.0)                               # the row maximum lands on the largest code
    assert np.abs(y).max() <= 448.0
    deq = O.dequantize_fp8(q, s).numpy()
    x = X.double().numpy()
    # nearest e4m3: relative error <= 2^-4 for normals, absolute <= 2^-10 * scale below the first normal
    assert np.all(np.abs(deq - x) <= np.maximum(2.0 ** -4 * np.abs(x), 2.0 ** -10 * s[:, None]) * (1 + 1e-6))
    # the codes are the nearest code points of y (brute force over the table), within half a spacing
    pts = O.e4m3_values()[:127]
    nearest = np.abs(np.abs(y)[:, :, None] - pts[None, None, :]).min(axis=2)
    np.testing.assert_array_equal(np.abs(np.abs(O.e4m3_values()[q]) - np.abs(y)), nearest)
    assert np.all(nearest <= O.e4m3_half_ulp(y))
    qt, st, yt = O.quantize_fp8(X, per_tensor=True)
    assert st.shape == (1,) and st[0] == amax.max() / 448.0
    assert np.abs(O.e4m3_values()[qt]).max() == 448.0
    # a power-of-two rescaling of the input changes the scale, not the codes
    q2, s2, _ = O.quantize_fp8((X.float() * 4).to(torch.bfloat16), per_tensor=False)
    assert np.array_equal(q2, q) and np.array_equal(s2[amax > 0], s[amax > 0] * 4)


def test_e4m3_half_ulp_is_half_the_code_point_spacing():
    pts = O.e4m3_values()[:127]
    gaps = np.diff(pts)
    mid = 0.5 * (pts[:-1] + pts[1:])
    np.testing.assert_array_equal(O.e4m3_half_ulp(mid), 0.5 * gaps)               # every interval between code points
    assert O.e4m3_half_ulp(0.0) == 2.0 ** -10 and O.e4m3_half_ulp(1.0) == 2.0 ** -4 and O.e4m3_half_ulp(-300.0) == 16.0
