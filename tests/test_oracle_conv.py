"""Pins for the u32 -> float conversions of the oracle (reading CONV; PAPER.md:443-446 says only
"uniformly distributed in the interval [0, 1)").  Exact rational values, interval ends, and the
reason u * 2^-32 rounded to float is rejected."""
from fractions import Fraction

import numpy as np

import oracle

EDGE = [0, 1, 255, 256, 257, 0x7FFFFFFF, 0x80000000, 0xFFFFFF00, 0xFFFFFFFF, 3338197162]


def test_f32_is_exact_and_below_one():
    L = oracle.lib()
    for u in EDGE:
        f = L.o_u32_to_f32(u)
        assert Fraction(f) == Fraction(u >> 8, 2**24)
        assert 0.0 <= f < 1.0
    assert L.o_u32_to_f32(0xFFFFFFFF) == 1.0 - 2.0**-24
    # the rejected alternative: u * 2^-32 rounded to float reaches 1.0
    assert np.float32(0xFFFFFFFF * 2.0**-32) == np.float32(1.0)


def test_f64_is_exact():
    L = oracle.lib()
    for u in EDGE:
        d = L.o_u32_to_f64(u)
        assert Fraction(d) == Fraction(u, 2**32)
        assert 0.0 <= d < 1.0


def test_fill_dtypes_agree_with_scalar_conversions():
    L = oracle.lib()
    for gen, seed in (("lfsr113", 12345), ("mt19937", 5489), ("gm31", 1), ("gq58.3", 1)):
        u = oracle.State(gen, seed).fill(300)
        f = oracle.State(gen, seed).fill(300, "f32")
        d = oracle.State(gen, seed).fill(300, "f64")
        assert f.dtype == np.float32 and d.dtype == np.float64
        assert f.tolist() == [L.o_u32_to_f32(int(x)) for x in u]
        assert d.tolist() == [L.o_u32_to_f64(int(x)) for x in u]
    # MRG32K3A f32 is the generic conversion of z_n (reading M4)
    u = oracle.State("mrg32k3a", 12345).fill(300)
    f = oracle.State("mrg32k3a", 12345).fill(300, "f32")
    assert f.tolist() == [L.o_u32_to_f32(int(x)) for x in u]
