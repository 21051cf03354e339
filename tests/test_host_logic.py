"""CPU tests of libprand's host side (no GPU, no compute call).

  * the library loads and exports every function include/prand.h and include/prand_host.h declare;
  * step a0 -- the skip operators the host prepares -- applied here to
    a state with plain Python integers reaches the state the oracle's own jump reaches;
  * the seed states the host prepares equal the oracle's;
  * the MT19937 characteristic polynomial from the closed form of ref. [2] equals the oracle's
    Berlekamp-Massey result, and the polynomial product composes jumps;
  * the launch policy covers every row exactly once;
  * argument errors are reported without touching CUDA.
"""
import ctypes as C
import os
import random
import re

import numpy as np
import pytest

import oracle
import paper_1307_5869_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DISTS = [0, 1, 2, 3, 777, 2**20 + 1, 2**40, 3 * 2**64, 12345 << 76, (2**63 + 5) << 100]
GM = ["gm19", "gm29", "gm31", "gm55", "gm61", "gq58.1", "gq58.3", "gq58.4"]
GM_G = {"gm19": 2**19 - 1, "gm29": 2**29 - 3, "gm31": 2**31 - 1, "gm55": 16 * (2**51 - 129),
        "gm61": 2**61 - 1, "gq58.1": 2**29 * (2**29 - 3), "gq58.3": 2**29 * (2**29 - 3),
        "gq58.4": 2**29 * (2**29 - 3)}
M1, M2 = 2**32 - 209, 2**32 - 22853
LFSR_MASK = [0xFFFFFFFE, 0xFFFFFFF8, 0xFFFFFFF0, 0xFFFFFF80]


def declared_functions():
    names = []
    for hdr in ("prand.h", "prand_host.h"):
        text = open(os.path.join(ROOT, "include", hdr)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names += re.findall(r"\b(prand_[a-z0-9_]+)\s*\(", text)
    return sorted(set(names))


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert len(names) >= 25
    raw = C.CDLL(P.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"libprand.so does not export {n}"
    # and the binding knows each of them
    assert set(names) == set(P.EXPORTS)


def test_version_and_strerror():
    assert b"sm_100a" in P.lib().prand_version()
    assert P.lib().prand_strerror(0) == b"ok"
    for code in range(-9, 0):
        assert P.lib().prand_strerror(code) not in (b"ok", b"unknown error code")


def test_argument_errors_before_any_cuda_call():
    h = C.c_void_p()
    L = P.lib()
    assert L.prand_init(C.byref(h), 99, 1, 1, 1, 0, None) == -1          # bad generator
    assert L.prand_init(C.byref(h), 0, 12345, 0, 1, 0, None) == -2        # no streams
    assert L.prand_init(C.byref(h), 0, 100, 4, 1, 0, None) == -3          # LFSR113 seed < 128
    assert L.prand_init(C.byref(h), 1, 0, 4, 1, 0, None) == -3            # MRG32K3A seed 0
    assert L.prand_init(C.byref(h), 1, 2**32 - 1, 4, 1, 0, None) == -3    # MRG32K3A seed >= m2
    assert L.prand_init(C.byref(h), 2, 2**32, 4, 1, 0, None) == -3        # MT19937 seed >= 2^32
    assert L.prand_init(C.byref(h), 3, 2**19 - 1, 4, 1, 0, None) == -3    # GM19 seed = 0 mod g
    assert L.prand_init(C.byref(h), 0, 12345, 2**40, 2**40, 0, None) == -4  # s * mant overflows
    assert L.prand_init(C.byref(h), 2, 5489, 2581103, 1, 64, None) == -2   # MT19937: more than PRAND_MT19937_MAX_STREAMS
    assert L.prand_init(None, 0, 12345, 4, 1, 0, None) == -2
    assert h.value is None
    assert L.prand_generate_u32(None, None, 4, None) == -2
    assert L.prand_jump(None, 1, 0, None) == -2
    assert L.prand_free(None) == -2


@pytest.mark.parametrize("dist", DISTS)
def test_lfsr113_skip_operator_reaches_oracle_state(dist):
    op = np.frombuffer(P.prand_host_skip_op("lfsr113", dist), dtype=np.uint32).reshape(4, 32)
    for seed in (12345, 0xDEADBEEF):
        z = np.frombuffer(P.prand_host_seed_state("lfsr113", seed), dtype=np.uint32)
        got = []
        for c in range(4):
            r = 0
            for j in range(32):
                if (int(z[c]) >> j) & 1:
                    r ^= int(op[c, j])
            got.append(r & LFSR_MASK[c])
        want = np.frombuffer(oracle.State("lfsr113", seed).jump(dist).export(), dtype=np.uint32)
        assert got == want.tolist()


@pytest.mark.parametrize("dist", DISTS)
def test_mrg32k3a_skip_operator_reaches_oracle_state(dist):
    op = np.frombuffer(P.prand_host_skip_op("mrg32k3a", dist), dtype=np.uint32).astype(object)
    A, B = op[:9].reshape(3, 3), op[9:].reshape(3, 3)
    st = np.frombuffer(P.prand_host_seed_state("mrg32k3a", 12345), dtype=np.uint32).astype(object)
    x = [sum(A[i, j] * st[j] for j in range(3)) % M1 for i in range(3)]
    y = [sum(B[i, j] * st[3 + j] for j in range(3)) % M2 for i in range(3)]
    want = np.frombuffer(oracle.State("mrg32k3a", 12345).jump(dist).export(), dtype=np.uint32)
    assert x + y == want.tolist()


@pytest.mark.parametrize("gen", GM)
def test_gm_skip_operator_and_seed_state_reach_oracle_state(gen):
    g = GM_G[gen]
    dt = np.uint32 if g < 2**32 else np.uint64
    for seed in (1, 987654321987):
        if seed % g == 0:
            continue
        base = np.frombuffer(P.prand_host_seed_state(gen, seed), dtype=dt).astype(object)
        assert base.tolist() == np.frombuffer(oracle.State(gen, seed).export(), dtype=dt).tolist()
        for dist in DISTS:
            m = np.frombuffer(P.prand_host_skip_op(gen, dist), dtype=np.uint64).astype(object)
            got = []
            for i in range(len(base) // 2):
                xP, xN = base[2 * i], base[2 * i + 1]
                got += [(m[2] * xN + m[3] * xP) % g, (m[0] * xN + m[1] * xP) % g]
            want = np.frombuffer(oracle.State(gen, seed).jump(dist).export(), dtype=dt).tolist()
            assert got == want, (gen, seed, dist)


def test_mt19937_phi_closed_form_equals_oracle_minimal_polynomial():
    deg, phi = oracle.mt19937_charpoly()
    mine = np.frombuffer(P.prand_host_mt19937_phi(), dtype=np.uint64)
    assert deg == 19937
    assert np.array_equal(mine[:312], phi)
    assert sum(bin(int(w)).count("1") for w in mine) == 135     # 135 non-zero terms
    assert P.lib().prand_host_mt19937_phi_selfcheck() == 0      # what prand_init checks once per process


@pytest.mark.parametrize("dist", [0, 1, 5, 623, 624, 19937, 50000, 2**64, (2**40 + 5) << 64, 12345 << 3])
def test_mt19937_jump_polynomial_equals_oracle(dist):
    a = np.frombuffer(P.prand_host_skip_op("mt19937", dist), dtype=np.uint64)
    assert np.array_equal(a, oracle.mt19937_jump_poly(dist))


def test_mt19937_polynomial_product_composes_jumps():
    rng = random.Random(7)
    for _ in range(4):
        a, b = rng.randrange(1, 2**60), rng.randrange(1, 2**60) << rng.randrange(0, 80)
        pa, pb = P.prand_host_skip_op("mt19937", a), P.prand_host_skip_op("mt19937", b)
        prod = np.frombuffer(P.prand_host_mt19937_mulmod(pa, pb), dtype=np.uint64)
        assert np.array_equal(prod, oracle.mt19937_jump_poly(a + b))


def test_mt19937_precomputed_table_is_the_papers_and_equals_the_oracle():
    """x^v mod phi stored for v = 2^n (n = 0..511) and v = m 2^i (m = 15..24, i = 0..127),
    2496 bytes each, < 5 MB.  Every record is pinned: the first of each chain (x, x^15 .. x^24) and deep
    ones against the oracle's own square-and-multiply, every other record as the square of its predecessor
    by the polynomial product (itself pinned to the oracle above)."""
    entries = [(1, n) for n in range(512)] + [(m, i) for m in range(15, 25) for i in range(128)]
    assert len(entries) == 1792 and len(entries) * 2496 < 5 * 2**20
    recs = {}
    for m, i in entries:
        r = P.prand_host_mt19937_table(m << i)
        assert r is not None, (m, i)
        recs[(m, i)] = r
    # not tabulated: other odd parts, powers beyond the table
    for v in (3, 7 << 10, 25 << 127, 2**512, 13 << 3, 15 << 128):
        assert P.prand_host_mt19937_table(v) is None
    # 16 = 2^4, 20 2^i = 5 2^(i+2) ...: one distance, one polynomial, whichever chain names it
    assert recs[(16, 3)] == recs[(1, 7)] and recs[(24, 0)] == P.prand_host_mt19937_table(3 << 3)
    # anchors against the oracle
    for m, i in [(1, 0), (1, 1), (1, 64), (1, 511)] + [(m, 0) for m in range(15, 25)] + [(15, 64), (24, 127)]:
        assert np.array_equal(np.frombuffer(recs[(m, i)], dtype=np.uint64), oracle.mt19937_jump_poly(m << i)), (m, i)
    # every record is the square of its predecessor
    for m, i in entries:
        if i:
            assert P.prand_host_mt19937_mulmod(recs[(m, i - 1)], recs[(m, i - 1)]) == recs[(m, i)], (m, i)


def test_mt19937_seed_state_equals_oracle():
    mine = np.frombuffer(P.prand_host_seed_state("mt19937", 5489), dtype=np.uint32).copy()
    want = np.frombuffer(oracle.State("mt19937", 5489).export(), dtype=np.uint32)
    mine[0] &= 0x80000000
    assert np.array_equal(mine, want)


@pytest.mark.parametrize("gen", ["lfsr113", "mrg32k3a", "gm31", "gm61", "gq58.3", "mt19937"])
def test_plan_covers_all_rows(gen):
    for ns in (1, 5, 512, 1024, 65536, 2**20):
        for n in (1, 3, 64, 100, 4096, 2**20):
            for dt in ("u32", "f64"):
                cl, nc = P.prand_host_plan(gen, ns, n, dt, 148)
                assert nc >= 1 and cl >= 1
                assert (nc - 1) * cl < n <= nc * cl
                if nc > 1:
                    assert cl % 4 == 0 and gen != "mt19937"
    # enough streams and an integer-bound kernel: never chunk
    assert P.prand_host_plan("gm31", 2**20, 2048, "u32", 148) == (2048, 1)
    assert P.prand_host_plan("mrg32k3a", 2**20, 2048, "u32", 148) == (2048, 1)
    # the store-bound kernels (LFSR113, MRG32K3A f64) take sub-sections of 1024 rows in several waves (measured faster
    # than one wave of long ones), also when the streams alone would fill the GPU; short calls stay whole
    assert P.prand_host_plan("lfsr113", 2**20, 2048, "u32", 148) == (1024, 2)
    assert P.prand_host_plan("lfsr113", 2**20, 2047, "u32", 148) == (2047, 1)
    assert P.prand_host_plan("mrg32k3a", 65536, 16384, "f64", 148) == (1032, 16)       # C2 (whole groups of 12 rows)
    assert P.prand_host_plan("lfsr113", 1024, 2**20, "u32", 148) == (1024, 1024)
    # config 1 (1024 streams x 4096) must be cut to fill the GPU: small L2-resident outputs run one stream per
    # thread, so 1024 threads x 64 sub-sections of 64 rows (a second wave would cost a whole sub-section)
    assert P.prand_host_plan("lfsr113", 1024, 4096, "u32", 148) == (64, 64)
    # integer-bound generators keep one balanced wave: sub-sections fill 148 x 1024 threads, no more
    cl, nc = P.prand_host_plan("gm31", 1024, 2**20, "u32", 148)
    assert nc * 1024 <= 148 * 1024 < 2 * nc * 1024 and cl % 4 == 0


def test_section_plan_covers_the_array_exactly_once():
    """prand_generate_seq_* (PAPER.md:382): sections tile [0, length) with no gap, no empty section."""
    import ctypes as C
    for gen in ("lfsr113", "mrg32k3a", "mt19937", "gm61"):
        for length in (1, 31, 1024, 4999, 8 * 624 * 2, 10**6 + 7, 2**29, 2**33 + 5):
            S, L = C.c_uint64(), C.c_uint64()
            assert P.lib().prand_host_plan_sections(P.gen_id(gen), length, C.byref(S), C.byref(L)) == 0
            S, L = S.value, L.value
            assert S >= 1 and L >= 1 and L % 32 == 0
            assert (S - 1) * L < length <= S * L
            assert S <= (4 * 148 if gen == "mt19937" else 131072)    # MT19937: one CTA of four sections per SM
    assert P.lib().prand_host_plan_sections(0, 0, C.byref(C.c_uint64()), C.byref(C.c_uint64())) == -2
    # the plan of a device with another multiprocessor count (MT19937: four sections per multiprocessor)
    S, L = C.c_uint64(), C.c_uint64()
    for sms in (148, 132, 20):
        assert P.lib().prand_host_plan_sections_sm(P.gen_id("mt19937"), 2**29, sms, C.byref(S), C.byref(L)) == 0
        assert S.value <= 4 * sms < S.value + 4 and L.value % 32 == 0 and (S.value - 1) * L.value < 2**29 <= S.value * L.value
    a, b = C.c_uint64(), C.c_uint64()
    assert P.lib().prand_host_plan_sections(P.gen_id("mt19937"), 2**29, C.byref(a), C.byref(b)) == 0
    assert P.lib().prand_host_plan_sections_sm(P.gen_id("mt19937"), 2**29, 148, C.byref(S), C.byref(L)) == 0
    assert (a.value, b.value) == (S.value, L.value)
    assert P.lib().prand_host_plan_sections_sm(0, 100, 0, C.byref(S), C.byref(L)) == -2


def test_mt19937_table_file_is_checked_when_it_is_loaded(tmp_path):
    """A table file of the right size whose records are not what they should be (stale layout, damaged bytes) must not
    be used: the library checks chain links with its own polynomial arithmetic at load and falls back to host
    arithmetic.  One process per case: the table is loaded once."""
    import subprocess
    import sys
    good = os.path.join(os.path.dirname(P.LIB_PATH), "mt19937_polys.bin")
    raw = bytearray(open(good, "rb").read())
    assert len(raw) == 1792 * 2496
    cases = {"good": bytes(raw)}
    flipped = bytearray(raw); flipped[255 * 2496 + 1000] ^= 0x10          # one bit in record x^(2^255)
    cases["bit flipped in a checked record"] = bytes(flipped)
    shifted = bytearray(raw); shifted[2 * 2496:] = raw[3 * 2496:] + raw[2 * 2496:3 * 2496]   # records from 2 on moved up by one
    cases["records shifted"] = bytes(shifted)
    rows = bytearray(raw); rows[512 * 2496:(512 + 128) * 2496] = raw[(512 + 128) * 2496:(512 + 256) * 2496]   # row m=15 holds m=16's
    cases["a row of another m"] = bytes(rows)
    code = ("import paper_1307_5869_b200 as P; "
            "print('TABLE', P.prand_host_mt19937_table(1 << 300) is not None, P.prand_host_mt19937_table(15 << 100) is not None)")
    for name, data in cases.items():
        path = tmp_path / "table.bin"
        path.write_bytes(data)
        env = dict(os.environ, PRAND_MT_TABLE=str(path), PYTHONPATH=ROOT)
        r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stderr
        used = "TABLE True True" in r.stdout
        assert used == (name == "good"), (name, r.stdout, r.stderr)
        if name != "good":
            assert "consistency check" in r.stderr


def test_bench_reference_arm_prints_the_contract_line():
    """bench.py --impl reference (this tier's reference arm = the oracle on the host cores) prints one
    JSON line with the contract's keys; no GPU is touched."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=300, cwd=root)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and "workload" in d["config"]


def test_gm_jump_coefficients_of_the_papers_relation():
    """x(2n+w) = k_n x(n+w) - q_n x(w).  The library's (k_n, q_n) (Lucas ladder by
    eq. 3-4) must be the trace and determinant of the n-th power of the companion matrix (the skip
    operator, computed by matrix powers), reproduce eq. 3, and drive the oracle's orbit by eq. 2."""
    import ctypes as C
    params = {"gm19": (15, 28, 2**19 - 1), "gm61": (24, 74, 2**61 - 1), "gm55": (256, 176, 16 * (2**51 - 129)),
              "gq58.3": (8, 48, 2**29 * (2**29 - 3))}
    def kq(gen, n):
        mant, log2 = P.split_dist(n)
        k, q = C.c_uint64(), C.c_uint64()
        assert P.lib().prand_host_gm_kq(P.gen_id(gen), mant, log2, C.byref(k), C.byref(q)) == 0
        return k.value, q.value
    for gen, (k, q, g) in params.items():
        assert kq(gen, 1) == (k % g, q % g)
        for n in (2, 3, 7, 1000, 2**26, 5 * 2**33, 3 * 2**70):
            kn, qn = kq(gen, n)
            m = np.frombuffer(P.prand_host_skip_op(gen, n), dtype=np.uint64).astype(object)
            assert kn == (m[0] + m[3]) % g and qn == (m[0] * m[3] - m[1] * m[2]) % g, (gen, n)
            assert qn == pow(q, n, g)
            k2, q2 = kq(gen, 2 * n)
            assert k2 == (kn * kn - 2 * qn) % g and q2 == qn * qn % g          # eq. 3
        # eq. 2 on the oracle's orbit (seed 1): x(2n+w) = k_n x(n+w) - q_n x(w)
        n, w = 12345, 678
        kn, qn = kq(gen, n)
        xw = oracle.gm_orbit(gen, 1, w)[0]
        xnw = oracle.gm_orbit(gen, 1, n + w)[0]
        x2nw = oracle.gm_orbit(gen, 1, 2 * n + w)[0]
        assert x2nw == (kn * xnw - qn * xw) % g
