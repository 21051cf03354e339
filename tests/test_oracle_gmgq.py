"""Pins for the GM/GQ oracle (oracle/gmgq.c) -- CPU only.

  * Table 2: the companion matrix of (k, q) has exact multiplicative order
    p^2 - 1 modulo the odd prime part p of g, and p^2 - 1 reproduces every printed period;
  * the paper's jump relations, eq. 2 with coefficients from eq. 3 (doubling) *and* eq. 4
    (linear recurrence), as identities on orbit points produced by the oracle;
  * a Lucas-sequence binary ladder (textbook identities U_{2n} = U_n V_n, V_{2n} = V_n^2 - 2Q^n,
    ...) as an independent algorithm for w(n), against the oracle's matrix power;
  * jump(n) == n single steps; composition; block splitting is positional;
  * the digit / packing rule (reading G2) re-evaluated with exact rationals on exported states,
    including the GM29 case where floor(2x/g) differs from a shift;
  * the seeding layout (reading G3) and its capacity arithmetic against Tables 2, 4 and 5.
"""
import ctypes
import random
from fractions import Fraction

import numpy as np
import pytest

import oracle
from test_oracle_mrg32k3a import factorize, is_probable_prime

# name: (k, q, g, v, s, d, printed period, odd prime part p)
TABLE = {
    "gm19": (15, 28, 2**19 - 1, 1, 32, 32, "2.7e+11", 2**19 - 1),
    "gm29": (4, 2, 2**29 - 3, 1, 32, 52, "2.8e+17", 2**29 - 3),
    "gm31": (11, 14, 2**31 - 1, 1, 32, 56, "4.6e+18", 2**31 - 1),
    "gm55": (256, 176, 16 * (2**51 - 129), 4, 8, 98, "5.1e+30", 2**51 - 129),
    "gm61": (24, 74, 2**61 - 1, 1, 32, 116, "5.3e+36", 2**61 - 1),
    "gq58.1": (8, 48, 2**29 * (2**29 - 3), 1, 32, 52, "2.8e+17", 2**29 - 3),
    "gq58.3": (8, 48, 2**29 * (2**29 - 3), 3, 12, 54, "2.8e+17", 2**29 - 3),
    "gq58.4": (8, 48, 2**29 * (2**29 - 3), 4, 8, 54, "2.8e+17", 2**29 - 3),
}
GENS = list(TABLE)


def words(gen, blob):
    g = TABLE[gen][2]
    return np.frombuffer(blob, dtype=np.uint32 if g < 2**32 else np.uint64).astype(object).tolist()


def lucas_w(k, q, g, seed, n):
    """w(n), w(n+1) for w(0)=0, w(1)=seed via the binary Lucas ladder on (U_m, U_{m+1}, Q^m).

    U_{2m} = U_m (2 U_{m+1} - k U_m), U_{2m+1} = U_{m+1}^2 - q U_m^2,
    U_{2m+2} = U_{m+1} (k U_{m+1} - 2 q U_m)      (all mod g); w(n) = seed * U_n."""
    u0, u1 = 0, 1
    for bit in bin(n)[2:] if n else "":
        a = u0 * (2 * u1 - k * u0) % g
        b = (u1 * u1 - q * u0 * u0) % g
        c = u1 * (k * u1 - 2 * q * u0) % g
        u0, u1 = (b, c) if bit == "1" else (a, b)
    return seed * u0 % g, seed * u1 % g


@pytest.mark.parametrize("gen", GENS)
def test_parameters_match_table2_and_periods(gen):
    k, q, g, v, s, d, printed, p = TABLE[gen]
    P = oracle.lib()

    class Par(ctypes.Structure):
        _fields_ = [("k", ctypes.c_uint64), ("q", ctypes.c_uint64), ("g", ctypes.c_uint64),
                    ("v", ctypes.c_uint), ("s", ctypes.c_uint), ("d", ctypes.c_uint)]
    par = Par()
    assert P.o_gm_params_get(oracle.gen_id(gen), ctypes.byref(par)) == 0
    assert (par.k, par.q, par.g, par.v, par.s, par.d) == (k, q, g, v, s, d)
    assert is_probable_prime(p) and g % p == 0 and (g // p) & (g // p - 1) == 0
    period = p * p - 1
    # the paper prints two significant digits (2.88e17 appears as 2.8e17, 5.07e30 as 5.1e30)
    assert abs(period / float(printed) - 1) < 0.03
    # exact order on the state of a stream far enough from the seed (past the 2-adic transient)
    st = oracle.State(gen, 1)
    st.fill(40)
    ref = st.export()
    assert st.copy().jump(period).export() == ref
    for r in sorted(factorize(period)):
        assert st.copy().jump(period // r).export() != ref, r
    # ensemble points sit on one orbit at disjoint offsets: (s+1) D < period  (G3)
    assert (s + 1) * 2**d < period


@pytest.mark.parametrize("gen", GENS)
def test_paper_eqs_2_3_4(gen):
    k, q, g, *_ = TABLE[gen]
    rng = random.Random(hash(gen) & 0xFFFF)
    x = lambda n: oracle.gm_orbit(gen, 1, n)[0]     # noqa: E731  x^(n) of the base orbit
    # eq. 4: k_0 = 2, k_1 = k, k_{n+1} = k k_n - q k_{n-1}; q_n = q^n
    ks = [2, k % g]
    for n in range(2, 70):
        ks.append((k * ks[-1] - q * ks[-2]) % g)
    for n in range(1, 70):
        qn = pow(q, n, g)
        for w in (0, 1, 5, rng.randrange(1 << 40)):
            assert x(2 * n + w) == (ks[n] * x(n + w) - qn * x(w)) % g, (n, w)
    # eq. 3: doubling k_{2n} = k_n^2 - 2 q_n, q_{2n} = q_n^2, for n = 2^i up to 2^100
    kn, qn, n = k % g, q % g, 1
    for i in range(100):
        for w in (0, 3, rng.randrange(1 << 64)):
            assert x(2 * n + w) == (kn * x(n + w) - qn * x(w)) % g, (i, w)
        kn, qn, n = (kn * kn - 2 * qn) % g, qn * qn % g, 2 * n
    # the consequence printed under eq. 2: x^(4n) = (k_n^2 - 2 q_n) x^(2n) - q_n^2 x^(0)
    n = 12345
    kn, qn = ks_n(k, q, g, n), pow(q, n, g)
    assert x(4 * n) == ((kn * kn - 2 * qn) * x(2 * n) - qn * qn * x(0)) % g


def ks_n(k, q, g, n):
    a, b = 2, k % g
    for _ in range(n):
        a, b = b, (k * b - q * a) % g
    return a


@pytest.mark.parametrize("gen", GENS)
def test_orbit_against_lucas_ladder(gen):
    k, q, g, *_ = TABLE[gen]
    rng = random.Random(5)
    for seed in (1, 2, 987654321 % g or 1):
        for n in [0, 1, 2, 3, 17, 1 << 32, (1 << 116) + 5] + [rng.randrange(1 << 120) for _ in range(6)]:
            assert oracle.gm_orbit(gen, seed, n) == lucas_w(k, q, g, seed, n), (seed, n)
    # seed 1: w(2n) = w(n) k_n  (U_2n = U_n V_n)
    n = 1000
    assert oracle.gm_orbit(gen, 1, 2 * n)[0] == oracle.gm_orbit(gen, 1, n)[0] * ks_n(k, q, g, n) % g


@pytest.mark.parametrize("gen", GENS)
def test_seeding_layout_g3(gen):
    k, q, g, v, s, d, *_ = TABLE[gen]
    for seed, P in ((1, 0), (1, 12345), (77, 3 << 40)):
        got = words(gen, oracle.State(gen, seed).jump(P).export())
        assert len(got) == 2 * s
        for i in range(s):
            assert (got[2 * i], got[2 * i + 1]) == lucas_w(k, q, g, seed, P + (i + 1) * 2**d), i
    with pytest.raises(ValueError):
        oracle.State(gen, 0)
    with pytest.raises(ValueError):
        oracle.State(gen, g)


@pytest.mark.parametrize("gen", GENS)
def test_jump_equals_single_steps_and_composes(gen):
    rng = random.Random(11)
    for n in [0, 1, 2, 15, 16, 1000] + [rng.randrange(1, 5000) for _ in range(3)]:
        a = oracle.State(gen, 1).jump(n)
        b = oracle.State(gen, 1)
        b.fill(n)
        assert a.export() == b.export(), n
        assert a.fill(5).tolist() == b.fill(5).tolist()
    a, b = rng.randrange(1 << 100), rng.randrange(1 << 100)
    assert oracle.State(gen, 3).jump(a).jump(b).export() == oracle.State(gen, 3).jump(a + b).export()


def pack(gen, state_words):
    """Reading G2 with exact rationals: digit_i = floor(2^v x_i / g), word = sum digit_i 2^(v i);
    GQ58.3: points 0..9 three bits at 3i, points 10, 11 one bit at 30, 31."""
    k, q, g, v, s, *_ = TABLE[gen]
    word = 0
    for i in range(s):
        xn = state_words[2 * i + 1]
        vi, pos = v, v * i
        if gen == "gq58.3" and i >= 10:
            vi, pos = 1, 30 + (i - 10)
        digit = int(Fraction(2**vi * xn, g))       # floor for non-negative rationals
        assert 0 <= digit < 2**vi
        word |= digit << pos
    return word


@pytest.mark.parametrize("gen", GENS)
def test_output_packing_g2(gen):
    k, q, g, v, s, *_ = TABLE[gen]
    st = oracle.State(gen, 1)
    for _ in range(200):
        before = words(gen, st.export())
        out = int(st.fill(1)[0])
        after = words(gen, st.export())
        for i in range(s):       # eq. 1 on every point
            assert after[2 * i] == before[2 * i + 1]
            assert after[2 * i + 1] == (k * before[2 * i + 1] - q * before[2 * i]) % g
        assert out == pack(gen, after)
    assert s * v == 32 or gen == "gq58.3"


def test_mersenne_digit_is_a_shift_but_gm29_is_not():
    # inject states whose next value is a chosen target: xN = 0, xP = -target / q mod g
    for gen, targets in (("gm19", [0, 2**18 - 1, 2**18, 2**19 - 2]),
                         ("gm31", [0, 2**30 - 1, 2**30, 2**31 - 2]),
                         ("gm61", [0, 2**60 - 1, 2**60, 2**61 - 2]),
                         ("gm29", [0, 2**28 - 2, 2**28 - 1, 2**28, 2**29 - 4])):
        k, q, g, v, s, *_ = TABLE[gen]
        dt = np.uint32 if g < 2**32 else np.uint64
        for t in targets:
            xp = (-t * pow(q, -1, g)) % g
            canon = np.array([xp, 0] * s, dtype=dt).tobytes()
            out = int(oracle.State(gen, 1).load(canon).fill(1)[0])
            want_bit = 1 if 2 * t >= g else 0
            assert out == (0xFFFFFFFF if want_bit else 0), (gen, t)
            if gen != "gm29":
                assert want_bit == t >> (g.bit_length() - 1)
    # GM29: x = 2^28 - 1 has digit 1 although x >> 28 == 0
    assert 2 * (2**28 - 1) >= 2**29 - 3 and (2**28 - 1) >> 28 == 0


@pytest.mark.parametrize("gen", ["gm55", "gq58.1", "gq58.3", "gq58.4"])
def test_two_adic_part_dies_out(gen):
    k, q, g, v, s, d, _, p = TABLE[gen]
    t2 = g // p
    # base orbit from w(0)=0, w(1)=1: after at most 16 steps every value is a multiple of 2^t
    vals = [oracle.gm_orbit(gen, 1, n)[0] for n in range(0, 64)]
    assert any(x % t2 for x in vals[:16])
    assert all(x % t2 == 0 for x in vals[16:])
    # and on multiples of 2^t the recurrence is the mod-p recurrence on y = x / 2^t
    ys = [x // t2 for x in vals[16:]]
    for a, b, c in zip(ys, ys[1:], ys[2:]):
        assert c == (k * b - q * a) % p
    # every stream state (positions >= D) is already in that regime
    assert all(x % t2 == 0 for x in words(gen, oracle.State(gen, 1).export()))


@pytest.mark.parametrize("gen", GENS)
def test_block_splitting_is_positional(gen):
    L, n, S = 19, 12, 5
    base = oracle.State(gen, 1).fill(S * L + n)
    out, states = oracle.streams(gen, 1, 0, S, L, n)
    for s_ in range(S):
        assert out[:, s_].tolist() == base[s_ * L: s_ * L + n].tolist()
        ref = oracle.State(gen, 1)
        ref.fill(s_ * L + n)
        assert states[s_].tobytes() == ref.export()


def test_capacity_of_the_chosen_block_lengths():
    # SURVEY.md 8(c) "Block lengths for C5": n_streams * L <= D keeps the points of all streams
    # on disjoint arcs; L does not exceed the Table 4 maximum of an init
    # function, except GM19 whose Table 4 row allows only 1000 sequences.
    n_streams = 2**20
    table4_max_len = {"gm29": 8e7, "gm55": 1e10, "gq58.1": 8e7, "gq58.3": 8e7, "gq58.4": 8e7,
                      "gm31": 8e7, "gm61": 1e10}
    block = {"gm19": 2**12, "gm29": 2**26, "gm55": 2**33, "gq58.1": 2**26, "gq58.3": 2**26,
             "gq58.4": 2**26, "gm31": 2**26, "gm61": 2**33}
    for gen, L in block.items():
        d = TABLE[gen][5]
        assert n_streams * L <= 2**d
        if gen in table4_max_len:
            assert L <= table4_max_len[gen]


def test_survey_third_opinion_values():
    # SURVEY.md 8(c) lists values computed in a separate scratch derivation (seed 1, first three
    # outputs of stream 0 | stream 1).  Not the paper's; kept as an independent cross-derivation.
    third = {
        ("gm19", 2**12): ([2994590615, 3019518940, 4201298895], [2483044914, 1854305385, 3151763912]),
        ("gm31", 2**26): ([3555403096, 2451403557, 2667641793], [142307092, 1390721089, 3046757752]),
        ("gm61", 2**33): ([3515631361, 2706664175, 3339134718], [746210390, 2698838255, 2263237635]),
        ("gm29", 2**26): ([4201370427, 2811808363, 2194022335], [926816331, 1493886411, 811946122]),
        ("gm55", 2**33): ([674644288, 4212495748, 2250356304], [841985338, 2693629897, 3036025546]),
        ("gq58.1", 2**26): ([1170092968, 1324267196, 4084410975], [1227712532, 3262070834, 1830904734]),
        ("gq58.3", 2**26): ([1090712108, 1966235245, 933828485], [1127281625, 1640035984, 320639716]),
        ("gq58.4", 2**26): ([29302969, 948626091, 3025370139], [675229282, 3492766800, 254944920]),
    }
    for (gen, L), (s0, s1) in third.items():
        out, _ = oracle.streams(gen, 1, 0, 2, L, 3)
        assert out[:, 0].tolist() == s0 and out[:, 1].tolist() == s1
