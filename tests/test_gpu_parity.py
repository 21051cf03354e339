"""GPU parity tests: libprand (CUDA, through the C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): bit-exact for uint32 outputs and exported states; f32/f64 are
compared bit-exactly too (both sides convert an exactly representable integer with a power-of-two
scale, or one IEEE multiply for MRG32K3A's f64 -- DESIGN.md "Tolerance"), so the |d| <= 2^-24 / 2^-53
fallback is never needed.  Small cases compare every output of every stream at sizes that span
several thread groups / tiles with ragged tails; the BASELINE.json configurations run at full size in
the launch configuration bench.py times and are compared on sampled streams (all rows of each).
"""
import ctypes as C
import os

import numpy as np
import pytest

import oracle
import workloads
from workloads import Workload

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1307_5869_b200 as P  # noqa: E402

ALL_GENS = P.GENS
NPDT = {"u32": np.uint32, "f32": np.float32, "f64": np.float64}
BITS = {"u32": np.uint32, "f32": np.uint32, "f64": np.uint64}
CPU_THREADS = min(16, os.cpu_count() or 1)


def need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def as_bits(a: np.ndarray, dtype: str) -> np.ndarray:
    return np.ascontiguousarray(a).view(BITS[dtype])


def lib_run(w: Workload, first=0, pre_jump=0, calls=None):
    """Generate w on the GPU -> (out as numpy (n, ns), canonical state bytes, kernel name)."""
    g = P.Generator(w.gen, w.seed, w.n_streams, w.block_len, first_stream=first)
    if pre_jump:
        g.jump(pre_jump)
    parts = []
    for n in (calls or [w.n_per_stream]):
        parts.append(g.generate(n, w.dtype))
    torch.cuda.synchronize()
    out = torch.cat(parts, 0).cpu().numpy().view(NPDT[w.dtype])
    st, k = g.state(), g.last_kernel
    g.close()
    return out, st, k


def oracle_run(w: Workload, first=0, pre_jump=0):
    out, states = oracle.streams(w.gen, w.seed, first, w.n_streams, w.block_len, w.n_per_stream,
                                 w.dtype, threads=CPU_THREADS, pre_jump=pre_jump)
    return out, states.tobytes()


def assert_same(w, got, want, what="outputs"):
    gb, wb = as_bits(got, w.dtype), as_bits(want, w.dtype)
    if not np.array_equal(gb, wb):
        bad = np.argwhere(gb != wb)
        i, s = bad[0]
        raise AssertionError(f"{w.name} {w.gen}/{w.dtype}: {len(bad)} of {gb.size} {what} differ; first at "
                             f"row {i} stream {s}: got {got[i, s]!r} want {want[i, s]!r}")


def small_cases(gen):
    # (n_streams, n_per_stream, block_len): a ragged stream count (scalar store path), a count that is
    # a multiple of 4 but of no CTA size, rows that are no multiple of the unroll / tile height
    if gen == "mt19937":      # the oracle's per-stream polynomial costs ~1 s at 2^64: keep streams few
        return [(5, 700, 2**64), (37, 70, 1000), (64, 33, 12345)]
    return [(37, 53, workloads.BLOCK_LEN[gen]), (1000, 67, workloads.BLOCK_LEN[gen]), (260, 129, 3)]


@pytest.mark.parametrize("dtype", ["u32", "f32", "f64"])
@pytest.mark.parametrize("gen", ALL_GENS)
def test_every_output_and_state_matches_oracle(gen, dtype):
    need_gpu()
    for ns, n, L in small_cases(gen):
        w = Workload(f"small-{ns}x{n}", gen, workloads.SEED.get(gen, 1), ns, L, n, dtype)
        got, st, _ = lib_run(w)
        want, wst = oracle_run(w)
        assert_same(w, got, want)
        assert st == wst, f"{w.name} {gen}: exported states differ"


MT_CFG_KERNEL = {0: "mt19937_bgen<S=32>", 1: "mt19937_gen<S=8,T=104>", 2: "mt19937_gen<S=4,T=208,pair>",
                 3: "mt19937_cgen<CS=4>", 4: "mt19937_tgen<S=4,T=208,pair>", 5: "mt19937_tgen<S=8,T=104>",
                 6: "mt19937_wgen<CS=2>"}


@pytest.mark.parametrize("cfg", range(7))
def test_mt19937_every_kernel_configuration(cfg, monkeypatch):
    """Every (streams per CTA, word slices, barrier interval, pipe mix, cluster pairing / cluster
    gather / TMA tile stores) variant of the MT19937 generation kernel, over whole rounds of 624, several
    rounds and ragged tails, with stream counts that leave CTAs partly or wholly dead."""
    need_gpu()
    P.prand_debug_set("PRAND_MT_CFG", str(cfg))
    cases = [(5, [624, 1248, 1, 700], "u32"), (13, [2048], "f32"), (8, [1500, 623], "f64"), (70, [209, 1300], "u32")]
    if cfg == 3:      # the cluster-gather kernel takes 4-byte outputs and stream counts that are multiples of 4
        cases = [(4, [624, 1248, 1, 700], "u32"), (12, [2048], "f32"), (16, [1500, 623, 3000], "u32"),
                 (68, [209, 1300, 1872], "u32"), (36, [5000], "f32")]
    if cfg >= 4:      # TMA tile stores: stream counts that are multiples of 4, calls of at least one round
        cases = [(4, [624, 1248, 700, 4000], "u32"), (12, [2048], "f32"), (8, [1500, 625, 3121], "f64"),
                 (68, [1300, 1872], "u32"), (36, [5000], "f32"), (20, [3000, 6240], "f64")]
    if cfg >= 6:      # warp-per-stream cluster kernel: whole clusters of 8 streams
        cases = [(8, [624, 1248, 700, 4000], "u32"), (16, [2048], "f32"), (8, [1500, 625, 3121], "f64"),
                 (72, [1300, 15, 1872, 656], "u32"), (40, [5000], "f32"), (24, [3000, 6240], "f64"),
                 # > 20 turns of 640 rows in one call: the six staging buffers wrap three times and both tile buffers of
                 # every helper warp are reused ten times (the wait for the TMA store that last read a tile), ragged tail
                 (8, [640 * 21 + 333], "u32"), (16, [640 * 25 + 17, 640 * 13 + 1], "f64")]
    for ns, calls, dtype in cases:
        w = Workload(f"mt-cfg{cfg}", "mt19937", 5489, ns, 1000, sum(calls), dtype)
        got, st, kernel = lib_run(w, calls=calls)
        assert kernel == MT_CFG_KERNEL[cfg], kernel
        want, wst = oracle_run(w)
        assert_same(w, got, want)
        assert st == wst, f"cfg {cfg}: exported states differ"
    P.prand_debug_set("PRAND_MT_CFG", None)


@pytest.mark.parametrize("gen", ALL_GENS)
def test_successive_calls_continue_the_streams(gen):
    need_gpu()
    ns, L = (6, 2**64) if gen == "mt19937" else (132, workloads.BLOCK_LEN[gen])
    w = Workload("continue", gen, workloads.SEED.get(gen, 1), ns, L, 700, "u32")
    got, st, _ = lib_run(w, calls=[1, 0, 30, 600, 69])
    want, wst = oracle_run(w)
    assert_same(w, got, want)
    assert st == wst


@pytest.mark.parametrize("gen", ALL_GENS)
def test_prand_jump_advances_every_stream(gen):
    need_gpu()
    ns, L = (4, 2**64) if gen == "mt19937" else (68, workloads.BLOCK_LEN[gen])
    for steps in (1, 1000, 5 << 70):
        if gen == "gm19" and steps > 2**30:
            continue
        w = Workload("jump", gen, workloads.SEED.get(gen, 1), ns, L, 40, "u32")
        got, st, _ = lib_run(w, pre_jump=steps)
        want, wst = oracle_run(w, pre_jump=steps)
        assert_same(w, got, want)
        assert st == wst


@pytest.mark.parametrize("gen", [g for g in ALL_GENS if g != "mt19937"])
def test_sub_section_chunking_changes_nothing(gen, monkeypatch):
    """a stream's range cut into sections reached by jump-ahead yields the same numbers."""
    need_gpu()
    w = Workload("chunked", gen, workloads.SEED.get(gen, 1), 44, workloads.BLOCK_LEN[gen], 203, "f32")
    want, wst = oracle_run(w)
    gid = P.gen_id(gen)
    for chunk in (4, 8, 52, 200):
        P.prand_debug_set("PRAND_CHUNK_LEN", str(chunk))
        # the hook is in force: the launch policy cuts the first call's 150 rows into more than one sub-section
        clen, ncs = C.c_uint64(), C.c_uint64()
        assert P.lib().prand_host_plan(gid, w.n_streams, 150, 1, 148, C.byref(clen), C.byref(ncs)) == 0
        gran = 32 if gen == "lfsr113" else 12
        forced = -(-chunk // gran) * gran
        if forced < 150:
            assert clen.value == forced and ncs.value == -(-150 // forced) > 1, (clen.value, ncs.value)
        else:                                             # (200: longer than either call, one section again)
            assert ncs.value == 1
        got, st, _ = lib_run(w, calls=[150, 53])
        assert_same(w, got, want)
        assert st == wst
    P.prand_debug_set("PRAND_CHUNK_LEN", None)


@pytest.mark.parametrize("gen", ["lfsr113", "mrg32k3a", "mt19937", "gm29", "gm61", "gq58.3"])
def test_shard_holds_its_slice_of_the_global_family(gen):
    need_gpu()
    L = 2**64 if gen == "mt19937" else workloads.BLOCK_LEN[gen]
    first, ns = (5, 7) if gen == "mt19937" else (1029, 75)
    w = Workload("shard", gen, workloads.SEED.get(gen, 1), ns, L, 31, "u32")
    got, st, _ = lib_run(w, first=first)
    want, wst = oracle_run(w, first=first)
    assert_same(w, got, want)
    assert st == wst


@pytest.mark.parametrize("gen", ALL_GENS)
def test_state_roundtrip_through_the_host(gen):
    """the state is plain data; copied out and back in, generation continues from it."""
    need_gpu()
    ns, L = (3, 1000) if gen == "mt19937" else (21, workloads.BLOCK_LEN[gen])
    seed = workloads.SEED.get(gen, 1)
    a = P.Generator(gen, seed, ns, L)
    a.generate(77, "u32")
    blob = a.state()
    rest_a = a.generate(50, "u32").cpu().numpy()
    b = P.Generator(gen, seed, ns, 0)            # block_len 0: all streams identical, then overwritten
    b.set_state(blob)
    assert b.state() == blob
    rest_b = b.generate(50, "u32").cpu().numpy()
    assert np.array_equal(rest_a, rest_b)
    want, _ = oracle.streams(gen, seed, 0, ns, L, 127, "u32", threads=CPU_THREADS)
    assert np.array_equal(rest_a.view(np.uint32), want[77:])
    a.close(); b.close()


@pytest.mark.parametrize("gen", ["gm55", "gq58.1", "gq58.3", "gq58.4"])
def test_imported_states_inside_the_two_adic_transient(gen):
    """g = 2^t p: the library's own states are multiples of 2^t and run the mod-p kernels; an imported
    state need not be (any residue mod g is a state).  Such states take the plain mod-g kernels until
    they have advanced 16 steps; outputs and states must equal the oracle's throughout."""
    need_gpu()
    ns = 9
    g_mod = {"gm55": 16 * (2**51 - 129)}.get(gen, 2**29 * (2**29 - 3))
    s_pts = {"gm55": 8, "gq58.1": 32, "gq58.3": 12, "gq58.4": 8}[gen]
    rng = np.random.default_rng(7)
    words = rng.integers(0, g_mod, size=(ns, 2 * s_pts), dtype=np.uint64)
    words[0, :] = [1, 0] * s_pts                           # degenerate small values too
    words[1, :] = g_mod - 1
    blob = words.tobytes()
    g = P.Generator(gen, 1, ns, 0)
    g.set_state(blob)
    calls = [3, 5, 9, 40, 25]
    got = []
    for n in calls:
        got.append(g.generate(n, "u32").cpu().numpy().view(np.uint32))
        if n == 9:
            assert "plain" in g.last_kernel
    assert "plain" not in g.last_kernel                   # past the transient: the mod-p kernel
    got = np.concatenate(got, 0)
    st = g.state()
    g.close()
    per = 2 * s_pts * 8
    for s in range(ns):
        o = oracle.State(gen, 1).load(blob[s * per:(s + 1) * per])
        want = o.fill(sum(calls), "u32")
        assert np.array_equal(got[:, s], want), f"{gen}: stream {s} differs from the oracle"
        assert st[s * per:(s + 1) * per] == o.export()


@pytest.mark.parametrize("gen,dtype", [("lfsr113", "u32"), ("mrg32k3a", "f64"), ("gm31", "f32"), ("mt19937", "u32")])
def test_host_delivery_equals_device_fill(gen, dtype):
    """rng_generate_array_: same numbers, delivered to host memory."""
    need_gpu()
    ns, L = (6, 1000) if gen == "mt19937" else (300, workloads.BLOCK_LEN[gen])
    w = Workload("host", gen, workloads.SEED.get(gen, 1), ns, L, 90, dtype)
    want, _ = oracle_run(w)
    g = P.Generator(w.gen, w.seed, w.n_streams, w.block_len)
    got = g.generate_host(w.n_per_stream, dtype).numpy().view(NPDT[dtype])
    assert_same(w, got, want)
    pageable = torch.empty((w.n_per_stream, ns), dtype=got_dtype(dtype))
    g2 = P.Generator(w.gen, w.seed, w.n_streams, w.block_len)
    g2.generate_host(w.n_per_stream, dtype, out=pageable)
    assert_same(w, pageable.numpy().view(NPDT[dtype]), want)
    g.close(); g2.close()


@pytest.mark.parametrize("gen", ALL_GENS)
def test_single_sequence_fill_equals_the_serial_generator(gen):
    """PAPER.md:382, 402-404 (rng_generate_gpu_array_): the array is cut into sections reached by
    jump-ahead, and holds exactly the numbers the serial generator produces, for any length."""
    need_gpu()
    seed = workloads.SEED.get(gen, 1)
    lengths = [100000, 7, 40001] if gen != "mt19937" else [30000, 5, 12345]
    # (LFSR113, MRG32K3A and MT19937 write the contiguous layout in place, with one kernel per element size)
    for dtype in (["u32", "f32", "f64"] if gen in ("mrg32k3a", "lfsr113", "mt19937") else
                  ["u32", "f64"] if gen == "gm31" else ["u32"]):
        g = P.Generator(gen, seed, 1, 0)
        g.jump(3)
        got = [g.generate_seq(n, dtype).cpu().numpy().view(NPDT[dtype]) for n in lengths]
        tail = g.generate(9, dtype).cpu().numpy().view(NPDT[dtype])[:, 0]     # the stream has advanced
        if lengths[0] >= 8 * 1024:
            assert "transpose" not in g.last_kernel
        st = g.state()
        g.close()
        o = oracle.State(gen, seed).jump(3)
        want = o.fill(sum(lengths) + 9, dtype)
        gotall = np.concatenate(got + [tail])
        assert np.array_equal(gotall.view(BITS[dtype]), want.view(BITS[dtype])), f"{gen}/{dtype}"
        assert st == o.export()


@pytest.mark.parametrize("gen", ["lfsr113", "mrg32k3a", "gm31"])
def test_single_sequence_fill_with_other_section_counts(gen):
    """PRAND_SEQ_SECTIONS caps the number of sections a sequence fill is cut into (tuning hook): the numbers are defined
    by position, so any cut gives the serial generator's output and state."""
    need_gpu()
    seed, n = workloads.SEED.get(gen, 1), 300_007
    want = oracle.State(gen, seed).fill(n, "u32")
    wst = oracle.State(gen, seed).jump(n).export()
    for cap in ("3", "64", "100000"):
        P.prand_debug_set("PRAND_SEQ_SECTIONS", cap)
        S, L = C.c_uint64(), C.c_uint64()
        assert P.lib().prand_host_plan_sections(P.gen_id(gen), n, C.byref(S), C.byref(L)) == 0
        assert S.value == min(int(cap), -(-n // L.value)) and S.value <= n // 1024      # the cap is in force
        g = P.Generator(gen, seed, 1, 0)
        got = g.generate_seq(n, "u32").cpu().numpy().view(np.uint32)
        st = g.state()
        g.close()
        assert np.array_equal(got, want), (gen, cap)
        assert st == wst
    P.prand_debug_set("PRAND_SEQ_SECTIONS", None)


def test_single_sequence_fill_needs_one_stream():
    need_gpu()
    g = P.Generator("lfsr113", 12345, 2, 1000)
    buf = torch.empty(16, dtype=torch.int32, device="cuda")
    assert P.lib().prand_generate_seq_u32(g._h, buf.data_ptr(), 16, None) == -2
    g.close()


@pytest.mark.parametrize("gen", ALL_GENS)
def test_device_callable_api_matches_oracle_and_bulk_kernels(gen):
    """the generators are callable from a user's kernel on the library's state.
    The library's example kernel (include/prand_device.cuh, one thread per stream) must produce the
    oracle's numbers, leave the oracle's state, and interleave freely with the bulk kernels."""
    need_gpu()
    seed = workloads.SEED.get(gen, 1)
    ns, L = (5, 1000) if gen == "mt19937" else (70, workloads.BLOCK_LEN[gen])
    for dtype in ("u32", "f32", "f64"):
        g = P.Generator(gen, seed, ns, L)
        a = g.device_api_fill(21, dtype).cpu().numpy().view(NPDT[dtype])
        b = g.generate(30, dtype).cpu().numpy().view(NPDT[dtype])          # bulk kernel continues
        c = g.device_api_fill(13, dtype).cpu().numpy().view(NPDT[dtype])
        assert g.last_kernel == "devapi_example"
        st = g.state()
        g.close()
        w = Workload("devapi", gen, seed, ns, L, 64, dtype)
        want, wst = oracle_run(w)
        assert_same(w, np.concatenate([a, b, c], 0), want)
        assert st == wst


def test_set_state_refuses_words_the_kernels_cannot_take():
    """The hot loops assume canonical residues and live components (x < m1, y < m2, GM words < g, no LFSR113
    component stuck at zero): prand_set_state range-checks an imported state and changes nothing on failure."""
    need_gpu()
    def try_set(gen, mutate, dt):
        g = P.Generator(gen, workloads.SEED.get(gen, 1), 3, 1000)
        good = g.state()
        a = np.frombuffer(good, dtype=dt).copy()
        mutate(a)
        rc = P.lib().prand_set_state(g._h, a.tobytes(), len(good))
        assert g.state() == (good if rc else a.tobytes())
        g.close()
        return rc
    def put(i, v):
        def f(a):
            a[i] = v
        return f
    def zero(lo, hi):
        def f(a):
            a[lo:hi] = 0
        return f
    assert try_set("mrg32k3a", put(7, 2**32 - 209), np.uint32) == -2            # x word = m1
    assert try_set("mrg32k3a", put(4, 2**32 - 22853), np.uint32) == -2          # y word = m2
    assert try_set("mrg32k3a", zero(6, 9), np.uint32) == -2                     # x component all zero
    assert try_set("lfsr113", put(5, 7), np.uint32) == -2                       # component 2: top 29 bits zero
    assert try_set("gm31", put(3, 2**31 - 1), np.uint32) == -2                  # = g
    assert try_set("gm61", put(10, 2**61 - 1), np.uint64) == -2
    assert try_set("gq58.3", put(2, 2**29 * (2**29 - 3)), np.uint64) == -2
    assert try_set("mrg32k3a", put(7, 2**32 - 210), np.uint32) == 0             # m1 - 1 is a residue
    assert P.lib().prand_trim() == 0


@pytest.mark.parametrize("hook", [None, "win", "win2", "win4", "list", "multi"])
def test_mt19937_every_polynomial_application_kernel(hook):
    """Eq. 10 in all its kernels: the four-streams-per-CTA form with the polynomial as a
    kernel argument (tree levels of >= 2368 streams) and from device memory (prand_jump by a distance that is
    not tabulated), the one-stream window form with one, two and four slices and the position-list forms (hooks),
    the 39-CTA wide form of the first levels (no hook) and the 640-thread and 4-CTA split forms that take its place
    under the "list" hook.
    Sampled streams against the oracle."""
    need_gpu()
    ns, L, steps = 6000, 2**64, (2**40 + 12345) << 480
    P.prand_debug_set("PRAND_MT_APPLY", hook)
    try:
        g = P.Generator("mt19937", 5489, ns, L)
        g.jump(steps)
        got = g.generate(40, "u32").cpu().numpy().view(np.uint32)
        st = g.state()
        g.close()
    finally:
        P.prand_debug_set("PRAND_MT_APPLY", None)
    sb = oracle.state_bytes("mt19937")
    for s in (0, 1, 3, 6, 13, 2047, 2048, 4096, ns - 1):
        want, wst = oracle.streams("mt19937", 5489, s, 1, L, 40, "u32", pre_jump=steps)
        assert np.array_equal(got[:, s], want[:, 0]), (hook, s)
        assert st[s * sb:(s + 1) * sb] == wst.tobytes(), (hook, s)


@pytest.mark.parametrize("cfg", range(7))
def test_shared_memory_kernels_repeat_bit_for_bit(cfg):
    """compute-sanitizer is not available on this GPU pool, so races in the shared-memory MT19937 kernels (in-place
    circular windows, deferred tempering, split cluster barriers, cp.async state loads, DSMEM bulk copies) are hunted
    by repetition instead: every kernel variant runs eight times from the same state at a size that fills the GPU,
    and all runs must agree bit for bit with the first, which is checked against the oracle on sampled streams."""
    need_gpu()
    ns = {0: 4736, 1: 1184, 2: 592, 3: 592, 4: 592, 5: 1184, 6: 592}[cfg]   # 148 CTAs of 32 / 8 / 4 / 4 / 4 / 8 streams
    n = 624 * 9 + 77
    P.prand_debug_set("PRAND_MT_CFG", str(cfg))
    try:
        g = P.Generator("mt19937", 5489, ns, 2**64)
        start = g.state()
        first = None
        for rep in range(8):
            g.set_state(start)
            out = g.generate(n, "u32")
            assert g.last_kernel == MT_CFG_KERNEL[cfg]
            if first is None:
                first, first_state = out.clone(), g.state()
            else:
                assert torch.equal(out, first), f"run {rep} differs from run 0"
                assert g.state() == first_state
        g.close()
    finally:
        P.prand_debug_set("PRAND_MT_CFG", None)
    got = first.cpu().numpy().view(np.uint32)
    for s in (0, ns // 2 + 1, ns - 1):
        want, _ = oracle.streams("mt19937", 5489, s, 1, 2**64, n, "u32")
        assert np.array_equal(got[:, s], want[:, 0]), s


def test_mt19937_jumps_use_the_precomputed_polynomial_table():
    """tabulated distances (2^n, n < 512; m 2^i, m = 15..24, i < 128) are one application of a
    device-resident polynomial; other distances are applied term by term of their binary notation; distances
    outside the table, or everything under PRAND_MT_POLY=host, go through the host's polynomial arithmetic.
    All must reach the oracle's state."""
    need_gpu()
    cases = [(2**20, "mt19937_apply<table>"), (20 << 30, "mt19937_apply<table>"), (5, "mt19937_apply<table>"),
             (12345, "mt19937_apply<table>"), (3 << 500, "mt19937_apply<table>"), (1 << 600, "mt19937_apply"),
             ((2**40 + 1) << 480, "mt19937_apply")]
    for steps, kernel in cases:
        w = Workload("mt-table", "mt19937", 5489, 3, 2**64, 30, "u32")
        want, wst = oracle_run(w, pre_jump=steps)
        for host in (False, True):
            P.prand_debug_set("PRAND_MT_POLY", "host" if host else None)
            try:
                g = P.Generator("mt19937", 5489, 3, 2**64)
                g.jump(steps)
                assert g.last_kernel == ("mt19937_apply" if host else kernel), (steps, g.last_kernel)
                got = g.generate(30, "u32").cpu().numpy().view(np.uint32)
                st = g.state()
                g.close()
            finally:
                P.prand_debug_set("PRAND_MT_POLY", None)
            assert_same(w, got, want)
            assert st == wst


def test_lfsr113_table_method_equals_matrix_jumps_and_oracle():
    """PAPER.md:363-370 (section 5.3): the paper's own jump algorithm for LFSR113 -- 128 tables per stream
    built by eq. 9, one warp per stream -- as an alternate of the GF(2) matrix path (PRAND_LFSR_INIT=table):
    stream initialisation by block splitting and prand_jump must reach the same states."""
    need_gpu()
    for ns, L, jump in [(70, 2**40, 12345), (33, 3 * 2**33, 5 << 40), (5, 1, 1), (130, 777, 0)]:
        w = Workload("lfsr-table", "lfsr113", 12345, ns, L, 40, "u32")
        ref, rst, _ = lib_run(w, pre_jump=jump)
        P.prand_debug_set("PRAND_LFSR_INIT", "table")
        try:
            g = P.Generator("lfsr113", 12345, ns, L)
            assert g.last_kernel == "lfsr113_table_jump"
            if jump:
                g.jump(jump)
                assert g.last_kernel == "lfsr113_table_jump"
            got = g.generate(40, "u32").cpu().numpy().view(np.uint32)
            st = g.state()
            g.close()
        finally:
            P.prand_debug_set("PRAND_LFSR_INIT", None)
        want, wst = oracle_run(w, pre_jump=jump)
        assert_same(w, got, want)
        assert np.array_equal(got, ref) and st == rst == wst


@pytest.mark.parametrize("gen", ALL_GENS)
def test_device_side_init_by_skipahead_matches_prand_init(gen):
    """PAPER.md:484-511 (rng_dev_init_sequence_ / rng_dev_skipahead_ over device constant tables): a
    user-style kernel loads the base stream, skips s * block_len ahead with the table of
    prand_device_ops and generates -- the numbers of the block-split family of prand_init."""
    need_gpu()
    seed = workloads.SEED.get(gen, 1)
    ns, L = (6, 2**64) if gen == "mt19937" else (77, workloads.BLOCK_LEN[gen])
    for dtype in (["u32", "f32", "f64"] if gen in ("mrg32k3a", "mt19937", "gm55") else ["u32"]):
        g = P.Generator(gen, seed, 1, 0)
        before = g.state()
        got = g.device_api_init_fill(ns, L, 45, dtype).cpu().numpy().view(NPDT[dtype])
        assert g.last_kernel == "devapi_init_example"
        assert g.state() == before                      # the base stream is not modified
        g.close()
        w = Workload("devinit", gen, seed, ns, L, 45, dtype)
        want, _ = oracle_run(w)
        assert_same(w, got, want)


@pytest.mark.parametrize("gen", ALL_GENS)
def test_skip_per_step_generator(gen):
    """PAPER.md:226, Table 3: the sequence that outputs one number and jumps `stride` ahead."""
    need_gpu()
    seed = workloads.SEED.get(gen, 1)
    ns, L = (2, 1000) if gen == "mt19937" else (37, workloads.BLOCK_LEN[gen])
    for stride, n in ((1, 5), (2, 6), (3 * 2**20, 4), (2**40, 3)):
        if (gen == "gm19" and stride > 2**20) or (gen == "mt19937" and stride > 2**30):
            continue
        g = P.Generator(gen, seed, ns, L)
        got = g.generate_strided(n, stride, "u32").cpu().numpy().view(np.uint32)
        st = g.state()
        g.close()
        for s in range(ns):
            o = oracle.State(gen, seed).jump(s * L)
            for i in range(n):
                assert got[i, s] == o.copy().fill(1, "u32")[0], f"{gen}: stride {stride} row {i} stream {s}"
                o.jump(stride)
            per = len(st) // ns
            assert st[s * per:(s + 1) * per] == o.export()


@pytest.mark.parametrize("gen", ["gm61", "gm55"])
@pytest.mark.parametrize("limit", ["0", "0xC0000000"])
def test_optimistic_steps_fall_back_exactly(gen, limit, monkeypatch):
    """GM61 / GM55 run an optimistic modular step and redo a group of points with the exact step when
    the watched limb reaches a limit (probability ~2^-28 in production).  Lowering the limit makes the
    fallback run always ("0") or for a quarter of the points: the numbers must not change."""
    need_gpu()
    P.prand_debug_set("PRAND_GM_WATCH", limit)
    for lp in ("1", "4") if gen == "gm61" else ("1",):
        P.prand_debug_set("PRAND_GM_LP", lp)
        w = Workload("watch", gen, 1, 70, workloads.BLOCK_LEN[gen], 37, "u32")
        got, st, _ = lib_run(w, calls=[20, 17])
        want, wst = oracle_run(w)
        assert_same(w, got, want)
        assert st == wst
    P.prand_debug_set("PRAND_GM_WATCH", None)
    P.prand_debug_set("PRAND_GM_LP", None)


@pytest.mark.parametrize("dtype", ["u32", "f32"])
def test_mrg32k3a_integer_and_fp64_pipe_kernels_agree_with_the_oracle(dtype, monkeypatch):
    """With 4-byte outputs MRG32K3A's second component runs on the FP64 pipe (exact: every product and
    fused sum is an integer below 2^53); PRAND_MRG_INT selects the all-integer kernel.  Both must be
    the oracle's numbers, also from states whose words exceed 2^31."""
    need_gpu()
    w = Workload("mrg-pipes", "mrg32k3a", 12345, 260, 2**76, 203, dtype)
    want, wst = oracle_run(w)
    for hook in (None, "1"):
        if hook:
            P.prand_debug_set("PRAND_MRG_INT", hook)
        got, st, kernel = lib_run(w, calls=[100, 103])
        assert kernel == ("mrg32k3a_gen<V=4,int>" if hook else "mrg32k3a_gen<V=4>"), kernel
        assert_same(w, got, want)
        assert st == wst
    P.prand_debug_set("PRAND_MRG_INT", None)


@pytest.mark.parametrize("gen", ["gm19", "gm31", "gm55", "gm61", "gq58.1", "gq58.3"])
def test_gm_family_init_by_the_papers_relation_equals_matrix_jumps(gen, monkeypatch):
    """prand_init fills GM/GQ families of >= 64 streams with x(2n+w) = k_n x(n+w) - q_n x(w)
    (eq. 2-3); PRAND_GM_INIT=matrix keeps one matrix jump per stream.  Same states,
    for ragged counts and shards, and both equal the oracle's."""
    need_gpu()
    L = workloads.BLOCK_LEN[gen]
    for first, ns in ((0, 64), (0, 1000), (5, 777), (0, 4099)):
        g = P.Generator(gen, 1, ns, L, first_stream=first)
        st_tree = g.state()
        assert g.last_kernel == "gm_tree"
        g.close()
        P.prand_debug_set("PRAND_GM_INIT", "matrix")
        g = P.Generator(gen, 1, ns, L, first_stream=first)
        st_mat = g.state()
        assert g.last_kernel == "gm_jump"
        g.close()
        P.prand_debug_set("PRAND_GM_INIT", None)
        assert st_tree == st_mat, f"{gen}: tree init differs from matrix init (first {first}, ns {ns})"
    _, wst = oracle.streams(gen, 1, 5, 777, L, 0, "u32", threads=CPU_THREADS)
    assert st_tree[:0] == b"" and P.Generator(gen, 1, 777, L, first_stream=5).state() == wst.tobytes()


@pytest.mark.parametrize("nf", ["0", "10", "16"])
def test_gm31_points_on_the_fp64_pipe_are_exact(nf, monkeypatch):
    """GM31 steps 14 of its 32 points in double precision on the FP64 pipe (exact floor division by
    2^31 - 1); PRAND_GM31_NF selects other splits (0: all points on the integer pipes)."""
    need_gpu()
    P.prand_debug_set("PRAND_GM31_NF", nf)
    w = Workload("gm31-fp64", "gm31", 1, 300, workloads.BLOCK_LEN["gm31"], 101, "u32")
    got, st, kernel = lib_run(w, calls=[50, 51])
    want, wst = oracle_run(w)
    assert_same(w, got, want)
    assert st == wst
    assert ("fp64" in kernel) == (nf != "0")
    P.prand_debug_set("PRAND_GM31_NF", None)


def got_dtype(dtype):
    return {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[dtype]


def test_degenerate_sizes_and_errors():
    need_gpu()
    g = P.Generator("lfsr113", 12345, 1, 2**40)
    out = g.generate(1, "u32")
    assert int(out.view(torch.int32)[0, 0]) & 0xFFFFFFFF == 3338197162   # SURVEY.md 8(c) sample value
    g.generate(0, "u32")                                                   # no-op
    assert P.lib().prand_generate_u32(g._h, None, 5, None) == -2
    buf = torch.empty(8, dtype=torch.int32, device="cuda")
    assert P.lib().prand_generate_f64(g._h, buf.data_ptr() + 4, 1, None) == -2   # misaligned for f64
    assert P.lib().prand_get_state(g._h, buf.data_ptr(), 3) == -6
    g.close()
    # block_len 0: every stream is the base sequence
    g = P.Generator("mrg32k3a", 12345, 9, 0)
    o = g.generate(4, "u32").cpu().numpy()
    assert (o == o[:, :1]).all()
    g.close()


def test_fill_probe_writes_every_word():
    need_gpu()
    for n in (1, 4, 1023, 4096 + 3, 1 << 22):
        buf = torch.zeros(n + 4, dtype=torch.int32, device="cuda")
        P.prand_fill_u32(buf.data_ptr(), n, 0x5A5A5A5A)
        torch.cuda.synchronize()
        h = buf.cpu().numpy().view(np.uint32)
        assert (h[:n] == 0x5A5A5A5A).all() and (h[n:] == 0).all()


def test_launch_counter_counts_kernels():
    need_gpu()
    before = P.prand_launch_count()
    g = P.Generator("gm55", 1, 32, 2**33)                # < 64 streams: one jump launch initialises them
    g.generate(8, "u32"); g.generate(8, "f32")
    assert P.prand_launch_count() - before == 3          # init + two fills
    assert "gm55" in g.last_kernel
    g.close()
