"""Pins for the LFSR113 oracle (oracle/lfsr113.c) -- CPU only.

Each pin ties the oracle to something other than itself:
  * a literal bit-by-bit program of PAPER.md:355-359 (eqs. 7-8), with no word tricks;
  * jump(n) == n single steps (the plain definition of jump-ahead);
  * the period printed in Table 2: (2^31-1)(2^29-1)(2^28-1)(2^25-1) = 1.0e34,
    each component returning to itself after exactly 2^p - 1 steps and not after (2^p-1)/r;
  * eq. 9 on the bit sequence the oracle's words are cut from;
  * composition of jumps and the block-splitting definition.
"""
import random

import numpy as np
import pytest

import oracle

PARAMS = [(31, 6, 18), (29, 2, 2), (28, 13, 7), (25, 3, 13)]


def bit_level_outputs(seed: int, n_out: int):
    """Eq. 7: x_n = x_{n-p} + x_{n-p+q} mod 2; eq. 8: u_n = sum_{i=1..32} x_{ns+i-1} 2^-i.

    x_0..x_{p-1} are the top p bits of the seed word, MSB first (reading L1).  Output number j
    (0-based) of the seed state is u_{j+1} (reading L2: step, then output)."""
    words = [0] * (n_out + 1)
    for (p, q, s) in PARAMS:
        need = (n_out + 1) * s + 32
        x = [(seed >> (31 - i)) & 1 for i in range(p)]
        for n in range(p, need):
            x.append(x[n - p] ^ x[n - p + q])
        for n in range(n_out + 1):
            u = 0
            for i in range(1, 33):
                u |= x[n * s + i - 1] << (32 - i)
            words[n] ^= u
    return words[1:]


@pytest.mark.parametrize("seed", [12345, 0xDEADBEEF, 0x80000000, 0xFFFFFFFF, 128])
def test_word_form_equals_bit_level_definition(seed):
    n = 10000 if seed == 12345 else 1500
    got = oracle.State("lfsr113", seed).fill(n)
    assert got.tolist() == bit_level_outputs(seed, n)


def test_eq9_holds_on_the_bit_sequence():
    # eq. 9: x_n = x_{n-kp} + x_{n-kp+kq} for k = 2^e, checked on bits rebuilt from eq. 7.
    for (p, q, s) in PARAMS:
        x = [(12345 >> (31 - i)) & 1 for i in range(p)]
        for n in range(p, 40 * p):
            x.append(x[n - p] ^ x[n - p + q])
        for e in range(1, 5):
            k = 1 << e
            for n in range(k * p, len(x)):
                assert x[n] == x[n - k * p] ^ x[n - k * p + k * q]


def test_invalid_seeds_rejected():
    for bad in [0, 1, 7, 15, 127]:   # some component has all top-p bits zero
        with pytest.raises(ValueError):
            oracle.State("lfsr113", bad)
    oracle.State("lfsr113", 128)


def test_jump_equals_single_steps():
    rng = random.Random(113)
    ns = [0, 1, 2, 31, 32, 33, 777, 4096, 10**6] + [rng.randrange(1, 200000) for _ in range(12)]
    for n in ns:
        a = oracle.State("lfsr113", 12345).jump(n)
        b = oracle.State("lfsr113", 12345)
        b.fill(n)
        assert a.export() == b.export(), n
        assert a.fill(16).tolist() == b.fill(16).tolist(), n


def test_jump_composition():
    rng = random.Random(7)
    for _ in range(10):
        a, b = rng.randrange(1 << 90), rng.randrange(1 << 90)
        s1 = oracle.State("lfsr113", 0xC0FFEE11).jump(a).jump(b)
        s2 = oracle.State("lfsr113", 0xC0FFEE11).jump(a + b)
        assert s1.export() == s2.export()
        assert s1.fill(8).tolist() == s2.fill(8).tolist()


def test_period_matches_table2():
    # period 1.0e34 = product of the four component periods 2^p - 1.
    comp = [(1 << p) - 1 for (p, _, _) in PARAMS]
    full = comp[0] * comp[1] * comp[2] * comp[3]
    assert f"{full:.1e}" == "1.0e+34"
    prime_factors = {31: [2**31 - 1], 29: [233, 1103, 2089], 28: [3, 5, 29, 43, 113, 127],
                     25: [31, 601, 1801]}
    for (p, _, _) in PARAMS:   # the factor lists really are the factorisations
        prod = 1
        for r in prime_factors[p]:
            assert ((1 << p) - 1) % r == 0
            prod *= r
        assert prod == (1 << p) - 1
    base = oracle.State("lfsr113", 12345)
    base.fill(1)                                    # canonical after one step
    ref = np.frombuffer(base.export(), dtype=np.uint32)
    # whole period: identity
    assert base.copy().jump(full).export() == base.export()
    for c, (p, _, _) in enumerate(PARAMS):
        after = np.frombuffer(base.copy().jump(comp[c]).export(), dtype=np.uint32)
        assert after[c] == ref[c]                   # component c is back
        for r in prime_factors[p]:
            if comp[c] // r == 1:
                continue
            part = np.frombuffer(base.copy().jump(comp[c] // r).export(), dtype=np.uint32)
            assert part[c] != ref[c], (p, r)         # ... and not earlier: order is exactly 2^p-1


def test_export_masks_untrusted_low_bits():
    st = np.frombuffer(oracle.State("lfsr113", 0xFFFFFFFF).export(), dtype=np.uint32)
    assert st.tolist() == [0xFFFFFFFE, 0xFFFFFFF8, 0xFFFFFFF0, 0xFFFFFF80]
    # low bits of the seed do not influence any output (L1)
    a = oracle.State("lfsr113", 0xABCDEF80).fill(64)
    b = oracle.State("lfsr113", 0xABCDEF80 | 0x01).fill(64)   # bit 0 is outside every top-p window
    assert a.tolist() == b.tolist()


def test_block_splitting_is_positional():
    # stream s = base sequence advanced s*block_len, small block so that the
    # plain definition (stepping) can be run.
    L, n, S = 37, 50, 9
    base = oracle.State("lfsr113", 12345).fill(S * L + n)
    out, states = oracle.streams("lfsr113", 12345, 0, S, L, n)
    for s in range(S):
        assert out[:, s].tolist() == base[s * L: s * L + n].tolist()
        ref = oracle.State("lfsr113", 12345)
        ref.fill(s * L + n)
        assert states[s].tobytes() == ref.export()


def test_streams_threads_and_offsets_agree():
    full, st_full = oracle.streams("lfsr113", 12345, 0, 12, 1 << 40, 20)
    part, st_part = oracle.streams("lfsr113", 12345, 5, 7, 1 << 40, 20, threads=3)
    assert np.array_equal(full[:, 5:], part)
    assert np.array_equal(st_full[5:], st_part)


def test_survey_sample_values():
    """tests/golden/survey_8c_samples.txt: the first five outputs for seed 12345 x 4 from the
    surveyor's independent bit-level implementation of eqs. 7-8 (readings L1, L2: the seed's low bits are
    ignored, the first output is the first stepped word)."""
    import os
    lines = [l for l in open(os.path.join(os.path.dirname(__file__), "golden", "survey_8c_samples.txt")) if not l.startswith("#")]
    vals = {l.split(":")[0]: l.split(":")[1].split() for l in lines}
    got = oracle.State("lfsr113", 12345).fill(5, "u32")
    assert [int(v) for v in got] == [int(v) for v in vals["lfsr113 seed=12345 u32"]]
