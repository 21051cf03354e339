"""Pins for the MRG32K3A oracle (oracle/mrg32k3a.c) -- CPU only.

  * the period printed in Table 2: 3.1e57 = (m1^3-1)(m2^3-1)/2, with A of exact
    order m1^3-1 and B of exact order m2^3-1 -- a wrong constant a, b, c, d, m1 or m2, a wrong
    sign or a transposed matrix (eq. 6) breaks full order;
  * the scalar three-term recurrences written out from eq. 5-6 with Python integers;
  * jump(n) == n single steps, composition, block splitting;
  * the f64 map (reading M3): exact rational value, open interval (0,1), z = 0 special case.
"""
import math
import random
from fractions import Fraction

import numpy as np
import pytest

import oracle

M1 = 2**32 - 209
M2 = 2**32 - 22853
A, B_, C_, D = 1403580, -810728, 527612, -1370589


def is_probable_prime(n: int) -> bool:
    if n < 2:
        return False
    for p in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):
        if n % p == 0:
            return n == p
    d, r = n - 1, 0
    while d % 2 == 0:
        d //= 2
        r += 1
    for a in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):
        x = pow(a, d, n)
        if x in (1, n - 1):
            continue
        for _ in range(r - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def pollard_rho(n: int) -> int:
    if n % 2 == 0:
        return 2
    rng = random.Random(n)
    while True:
        c, y, d = rng.randrange(1, n), rng.randrange(0, n), 1
        x = y
        while d == 1:
            x = (x * x + c) % n
            y = (y * y + c) % n
            y = (y * y + c) % n
            d = math.gcd(abs(x - y), n)
        if d != n:
            return d


def factorize(n: int) -> set:
    if n == 1:
        return set()
    if is_probable_prime(n):
        return {n}
    d = pollard_rho(n)
    return factorize(d) | factorize(n // d)


def scalar_sequence(seed: int, n: int):
    """x_{n+1} = a x_{n-1} + b x_{n-2} mod m1, y_{n+1} = c y_n + d y_{n-2} mod m2 (row 0 of eq. 6)."""
    x = [seed, seed, seed]   # x_n, x_{n-1}, x_{n-2}
    y = [seed, seed, seed]
    zs = []
    for _ in range(n):
        xn = (A * x[1] + B_ * x[2]) % M1
        yn = (C_ * y[0] + D * y[2]) % M2
        x = [xn, x[0], x[1]]
        y = [yn, y[0], y[1]]
        zs.append((xn - yn) % M1)
    return zs, x, y


def test_scalar_recurrence():
    zs, x, y = scalar_sequence(12345, 5000)
    st = oracle.State("mrg32k3a", 12345)
    assert st.fill(5000).tolist() == zs
    assert np.frombuffer(st.export(), dtype=np.uint32).tolist() == x + y


def test_exact_order_matches_printed_period():
    # PAPER.md:246 prints 3.1e57.
    per = (M1**3 - 1) * (M2**3 - 1) // 2
    assert f"{per:.1e}" == "3.1e+57"
    assert is_probable_prime(M1) and is_probable_prime(M2)
    st = oracle.State("mrg32k3a", 12345)
    st.fill(3)
    ref = np.frombuffer(st.export(), dtype=np.uint32)
    for which, m in ((0, M1), (1, M2)):
        order = m**3 - 1
        back = np.frombuffer(st.copy().jump(order).export(), dtype=np.uint32)
        assert back[3 * which: 3 * which + 3].tolist() == ref[3 * which: 3 * which + 3].tolist()
        for r in sorted(factorize(order)):
            part = np.frombuffer(st.copy().jump(order // r).export(), dtype=np.uint32)
            assert part[3 * which: 3 * which + 3].tolist() != ref[3 * which: 3 * which + 3].tolist(), r
    # the combined state returns after lcm = (m1^3-1)(m2^3-1)/2 (gcd of the two orders is 2)
    assert math.gcd(M1**3 - 1, M2**3 - 1) == 2
    assert st.copy().jump(per).export() == st.export()
    assert st.copy().jump(per // 2).export() != st.export()


def test_order_is_a_property_of_the_matrix_not_of_one_vector():
    # exact order on three independent start vectors (a basis), so A^order = I as a matrix
    for seed in (1, 2, 4294944442):
        st = oracle.State("mrg32k3a", seed)
        st.fill(seed % 5)
        assert st.copy().jump(M1**3 - 1).export()[:12] == st.export()[:12]
        assert st.copy().jump(M2**3 - 1).export()[12:] == st.export()[12:]


def test_jump_equals_single_steps():
    rng = random.Random(32)
    for n in [0, 1, 2, 3, 1000, 10**6] + [rng.randrange(1, 300000) for _ in range(10)]:
        a = oracle.State("mrg32k3a", 12345).jump(n)
        b = oracle.State("mrg32k3a", 12345)
        b.fill(n)
        assert a.export() == b.export(), n
        assert a.fill(8).tolist() == b.fill(8).tolist()


def test_jump_composition_large():
    rng = random.Random(3)
    for _ in range(10):
        a, b = rng.randrange(1 << 150), rng.randrange(1 << 150)
        s1 = oracle.State("mrg32k3a", 777).jump(a).jump(b)
        s2 = oracle.State("mrg32k3a", 777).jump(a + b)
        assert s1.export() == s2.export()


def test_invalid_seed():
    for bad in (0, M2, M2 + 5, 2**32):
        with pytest.raises(ValueError):
            oracle.State("mrg32k3a", bad)


def test_f64_map_reading_m3():
    L = oracle.lib()
    norm = Fraction(1, M1 + 1)
    for z in [1, 2, 12345, 545508589, M1 - 1, M1 // 2]:
        got = L.o_mrg32k3a_to_f64(z)
        assert 0.0 < got < 1.0
        # one correctly rounded multiply by the double nearest to 1/(m1+1)
        assert got == z * 2.328306549295727688e-10
        assert abs(Fraction(got) - z * norm) < Fraction(1, 2**52)
    assert L.o_mrg32k3a_to_f64(0) == M1 * 2.328306549295727688e-10 < 1.0
    assert abs(Fraction(2.328306549295727688e-10) - norm) < norm / 2**52
    zs = oracle.State("mrg32k3a", 12345).fill(100)
    fs = oracle.State("mrg32k3a", 12345).fill(100, "f64")
    assert fs.tolist() == [L.o_mrg32k3a_to_f64(int(z)) for z in zs]
    assert all(0 <= int(z) < M1 for z in zs)


def test_block_splitting_is_positional():
    L, n, S = 53, 40, 7
    base = oracle.State("mrg32k3a", 12345).fill(S * L + n)
    out, states = oracle.streams("mrg32k3a", 12345, 0, S, L, n)
    for s in range(S):
        assert out[:, s].tolist() == base[s * L: s * L + n].tolist()
    full, st_full = oracle.streams("mrg32k3a", 12345, 0, 10, 1 << 76, 12, "f64")
    part, st_part = oracle.streams("mrg32k3a", 12345, 4, 6, 1 << 76, 12, "f64", threads=2)
    assert np.array_equal(full[:, 4:], part) and np.array_equal(st_full[4:], st_part)


def test_survey_sample_values_pin_the_combination_sign():
    """tests/golden/survey_8c_samples.txt: the first outputs for seed 12345 x 6 from an
    independent implementation.  They fix reading M1 -- z = (x - y) mod m1, not (x + y) -- and the
    normalisation M3 (PAPER.md:347 is garbled on both)."""
    import os
    lines = [l for l in open(os.path.join(os.path.dirname(__file__), "golden", "survey_8c_samples.txt")) if not l.startswith("#")]
    vals = {l.split(":")[0]: l.split(":")[1].split() for l in lines}
    st = oracle.State("mrg32k3a", 12345)
    z = st.fill(5, "u32")
    assert [int(v) for v in z] == [int(v) for v in vals["mrg32k3a seed=12345 u32"]]
    x, y, z0 = (int(v) for v in vals["mrg32k3a seed=12345 first_x_y_z"])
    one = np.frombuffer(oracle.State("mrg32k3a", 12345).jump(1).export(), dtype=np.uint32)
    assert (int(one[0]), int(one[3])) == (x, y) and (x - y) % (2**32 - 209) == z0 and (x + y) % (2**32 - 209) != z0
    f = oracle.State("mrg32k3a", 12345).fill(1, "f64")[0]
    assert f"{f:.16f}" == vals["mrg32k3a seed=12345 f64_first"][0] and f == z0 / (2**32 - 208)
