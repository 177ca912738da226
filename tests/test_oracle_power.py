"""Pins of the oracle's power calculation: hand-computed values and exact integer arithmetic."""
import numpy as np

import oracle


def test_power_hand_values_and_rounding():
    v = np.array([[3, 4], [0, 0], [-5, 12], [-32768, -32768], [32767, 32767], [1, -1], [-32768, 0]], dtype=np.int16)
    p = oracle.power_i16(v)
    assert p.dtype == np.float32
    # 25, 0, 169, 2^31 (exact in fp32); 2 * 32767^2 = 2147352578 lies in [2^30, 2^31) where floats are 128 apart:
    # 2147352578 = 16776192 * 128 + 2 -> rounds down to 2147352576
    assert p.tolist() == [25.0, 0.0, 169.0, 2147483648.0, 2147352576.0, 2.0, 1073741824.0]


def test_power_matches_python_integers():
    g = np.random.default_rng(0)
    v = g.integers(-32768, 32768, size=(1000, 2)).astype(np.int16)
    p = oracle.power_i16(v)
    exact = [int(a) * int(a) + int(b) * int(b) for a, b in v.tolist()]          # unbounded Python integers
    assert all(float(np.float32(e)) == float(q) for e, q in zip(exact, p.tolist()))
    small = np.abs(v.astype(np.int64)).max(axis=1) < 2896                       # sums below 2^24: exact in fp32
    assert all(int(q) == e for e, q, s in zip(exact, p.tolist(), small.tolist()) if s)
