"""Pins for the MT19937 oracle (oracle/mt19937.c) -- CPU only.

  * BASELINE.json's check value: seed 5489 -> 10000th output = 4123659995 (tests/golden);
  * library routines: CPython's `random` (state injected, so it pins recurrence + tempering),
    numpy's MT19937 bit generator (seeding; `jumped()` = a 2^128 jump by an independent
    polynomial implementation) and libstdc++'s std::mt19937 incl. discard();
  * jump(v) == v single steps for v up to 10^6 (eq. 10);
  * phi: degree 19937, phi(A) W = 0 on every bit plane, and the period invariant
    x^(2^19937) = x (mod phi) computed here with Python integers (period
    4.3e6001 = 2^19937 - 1).
"""
import os
import random
import shutil
import subprocess

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_baseline_check_value():
    with open(os.path.join(GOLDEN, "mt19937_check.txt")) as f:
        fields = dict(line.split("=") for line in f.read().split() if "=" in line)
    seed, index, value = int(fields["seed"]), int(fields["output_number"]), int(fields["value"])
    out = oracle.State("mt19937", seed).fill(index)
    assert int(out[index - 1]) == value == 4123659995


def test_against_cpython_random_module():
    st = oracle.State("mt19937", 5489)
    key = np.frombuffer(st.export(), dtype=np.uint32).copy()
    key[0] = 5489                      # export zeroes the 31 unused bits; CPython wants the word
    r = random.Random()
    r.setstate((3, tuple(int(k) for k in key) + (624,), None))
    want = [r.getrandbits(32) for _ in range(3000)]
    assert st.fill(3000).tolist() == want


def test_against_numpy_seeding_and_stream():
    bg = np.random.MT19937()
    bg._legacy_seeding(20240229)
    key = bg.state["state"]["key"]
    mine = np.frombuffer(oracle.State("mt19937", 20240229).export(), dtype=np.uint32)
    assert mine[1:].tolist() == key[1:].tolist()
    assert mine[0] == key[0] & 0x80000000
    assert oracle.State("mt19937", 20240229).fill(2000).tolist() == bg.random_raw(2000).tolist()


def test_against_numpy_jumped_2_pow_128():
    # numpy ships its own precomputed polynomial for a 2^128 jump.  Its jumped key is a circular
    # buffer whose logical word i sits at key[(pos + i) % 624]; un-rotated it must be the window
    # x_{2^128}..x_{2^128+623} of the sequence whose x_0..x_623 is the seeded array.  Only the top
    # bit of word 0 belongs to the state (reading T2).
    for seed in (5489, 1):
        bg = np.random.MT19937()
        bg._legacy_seeding(seed)
        st = bg.jumped(1).state["state"]
        window = np.roll(st["key"], -int(st["pos"]))
        mine = np.frombuffer(oracle.State("mt19937", seed).jump(1 << 128).export(), dtype=np.uint32)
        assert mine[1:].tolist() == window[1:].tolist()
        assert mine[0] == window[0] & 0x80000000


@pytest.mark.skipif(shutil.which("g++") is None, reason="needs g++")
def test_against_libstdcxx(tmp_path):
    src = tmp_path / "m.cpp"
    src.write_text(
        "#include <random>\n#include <cstdio>\n#include <cstdlib>\n"
        "int main(int c,char**v){std::mt19937 g(strtoul(v[1],0,10));"
        "g.discard(strtoull(v[2],0,10));for(int i=0;i<8;i++)printf(\"%u\\n\",(unsigned)g());}\n")
    exe = tmp_path / "m"
    subprocess.check_call(["g++", "-O1", "-o", str(exe), str(src)])
    for seed, skip in [(5489, 0), (1, 12345), (4357, 700000)]:
        want = [int(x) for x in subprocess.check_output([str(exe), str(seed), str(skip)]).split()]
        assert oracle.State("mt19937", seed).jump(skip).fill(8).tolist() == want


def test_jump_equals_single_steps():
    rng = random.Random(19937)
    for v in [0, 1, 5, 623, 624, 625, 1000, 19936, 19937, 19938, 50000, 10**6] + \
             [rng.randrange(1, 400000) for _ in range(4)]:
        a = oracle.State("mt19937", 5489).jump(v)
        b = oracle.State("mt19937", 5489)
        b.fill(v)
        assert a.export() == b.export(), v
        assert a.fill(700).tolist() == b.fill(700).tolist(), v


def test_jump_composition():
    a, b = (1 << 64) + 12345, 3 << 70
    s1 = oracle.State("mt19937", 5489).jump(a).jump(b)
    s2 = oracle.State("mt19937", 5489).jump(a + b)
    assert s1.export() == s2.export()


def _phi_terms():
    deg, phi = oracle.mt19937_charpoly()
    val = 0
    for i, w in enumerate(phi):
        val |= int(w) << (64 * i)
    return deg, val


def test_charpoly_degree_and_annihilation():
    deg, phi = _phi_terms()
    assert deg == 19937 and phi.bit_length() == 19938 and phi & 1
    terms = [i for i in range(19938) if (phi >> i) & 1]
    # phi(A) W = 0: sum_i phi_i x_{t+i} = 0 for every word position t >= 1 and every bit plane;
    # sequence from numpy (library), not from the oracle
    bg = np.random.MT19937()
    bg._legacy_seeding(99)
    bg.random_raw(624)                       # now key = x_624..x_1247
    seq = []
    for _ in range(34):
        seq.append(bg.state["state"]["key"].copy())
        bg.random_raw(624)
    x = np.concatenate(seq)
    for t in (0, 1, 17, 600):
        acc = np.uint32(0)
        for e in terms:
            acc ^= x[t + e]
        assert acc == 0


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_period_invariant_x_pow_2_19937(tmp_path):
    # x^(2^19937) = x (mod phi)  <=>  every irreducible factor of phi has degree dividing the
    # prime 19937; with deg phi = 19937 and phi(0) = phi(1) = 1 this makes phi irreducible, and
    # 2^19937 - 1 prime then gives the period printed in PAPER.md:247 (4.3e6001).
    # The 19937 squarings run in tests/helpers/gf2_frobenius.c (own arithmetic, not the oracle's).
    deg, phi = _phi_terms()
    assert bin(phi).count("1") % 2 == 1 and phi & 1        # phi(1) = 1, phi(0) = 1
    low_terms = [i for i in range(19937) if (phi >> i) & 1]
    exe = tmp_path / "frob"
    subprocess.check_call(["gcc", "-O2", "-o", str(exe),
                           os.path.join(os.path.dirname(__file__), "helpers", "gf2_frobenius.c")])
    text = " ".join(str(v) for v in [deg] + low_terms)
    assert subprocess.check_output([str(exe)], input=text.encode()).split() == [b"1"]
    # negative control: dropping one term must break it
    text = " ".join(str(v) for v in [deg] + low_terms[:-1])
    assert subprocess.check_output([str(exe)], input=text.encode()).split() == [b"0"]
    # 2^19937 - 1 = 4.3e6001: log10 = 19937*log10(2) = 6001.63..., 10^0.6335 = 4.3
    import math
    lg = 19937 * math.log10(2)
    assert int(lg) == 6001 and f"{10 ** (lg - 6001):.1f}" == "4.3"


def test_jump_poly_is_x_pow_v_mod_phi():
    # small v: x^v itself; v = 19937: phi without its leading term
    deg, phi = _phi_terms()
    g = oracle.mt19937_jump_poly(100)
    val = sum(int(w) << (64 * i) for i, w in enumerate(g))
    assert val == 1 << 100
    g = oracle.mt19937_jump_poly(19937)
    val = sum(int(w) << (64 * i) for i, w in enumerate(g))
    assert val == phi ^ (1 << 19937)


def test_block_splitting_is_positional():
    L, n, S = 700, 30, 4
    base = oracle.State("mt19937", 5489).fill(S * L + n)
    out, states = oracle.streams("mt19937", 5489, 0, S, L, n)
    for s in range(S):
        assert out[:, s].tolist() == base[s * L: s * L + n].tolist()
    full, st_full = oracle.streams("mt19937", 5489, 0, 4, 1 << 64, 10, threads=4)
    part, st_part = oracle.streams("mt19937", 5489, 2, 2, 1 << 64, 10)
    assert np.array_equal(full[:, 2:], part) and np.array_equal(st_full[2:], st_part)
