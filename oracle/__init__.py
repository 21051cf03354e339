"""CPU oracle for the PRAND hot path -- TEST INFRASTRUCTURE ONLY.

Plain scalar C (``oracle/*.c``, compiled here with gcc) written from the paper's definitions
 and SURVEY.md section 8(c)'s readings.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It shares no code with ``paper_1307_5869_b200`` and never imports it.

This module only marshals arguments (ctypes + numpy); all arithmetic lives in the C files.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = ["lfsr113.c", "mrg32k3a.c", "mt19937.c", "gmgq.c", "driver.c"]
_LIB_PATH = os.path.join(_HERE, "_build", "liboracle.so")

GENS = ["lfsr113", "mrg32k3a", "mt19937", "gm19", "gm29", "gm31", "gm55", "gm61",
        "gq58.1", "gq58.3", "gq58.4"]
GEN_ID = {name: i for i, name in enumerate(GENS)}
DTYPES = {"u32": (0, np.uint32), "f32": (1, np.float32), "f64": (2, np.float64)}

_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/*.c into oracle/_build/liboracle.so (gcc -O2, no SIMD flags)."""
    srcs = [os.path.join(_HERE, s) for s in _SRC]
    deps = srcs + [os.path.join(_HERE, "oracle.h")]
    if not force and os.path.exists(_LIB_PATH):
        if os.path.getmtime(_LIB_PATH) >= max(os.path.getmtime(d) for d in deps):
            return _LIB_PATH
    os.makedirs(os.path.dirname(_LIB_PATH), exist_ok=True)
    tmp = _LIB_PATH + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra",
                           "-o", tmp] + srcs)
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def lib() -> C.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            L = C.CDLL(build())
            u8p, vp = C.c_char_p, C.c_void_p
            L.oracle_internal_bytes.restype = C.c_size_t
            L.oracle_internal_bytes.argtypes = [C.c_int]
            L.oracle_state_bytes.restype = C.c_size_t
            L.oracle_state_bytes.argtypes = [C.c_int]
            L.oracle_seed.argtypes = [C.c_int, C.c_uint64, vp]
            L.oracle_jump.argtypes = [C.c_int, vp, u8p, C.c_size_t]
            L.oracle_export.argtypes = [C.c_int, vp, vp]
            L.oracle_export.restype = None
            L.oracle_import.argtypes = [C.c_int, vp, vp]
            L.oracle_fill.argtypes = [C.c_int, vp, C.c_uint64, C.c_int, vp, C.c_uint64]
            L.oracle_streams.argtypes = [C.c_int, C.c_uint64, C.c_uint64, u8p, C.c_size_t,
                                         C.c_uint64, C.c_int, vp, C.c_uint64, C.c_uint64, vp]
            L.o_mt19937_charpoly.argtypes = [vp]
            L.o_mt19937_jump_poly.argtypes = [u8p, C.c_size_t, vp]
            L.o_mt19937_jump_poly.restype = None
            L.o_mt19937_apply_poly.argtypes = [vp, vp]
            L.o_mt19937_apply_poly.restype = None
            L.o_gm_orbit.argtypes = [C.c_int, C.c_uint64, u8p, C.c_size_t, vp, vp]
            L.o_gm_orbit.restype = None
            L.o_mrg32k3a_to_f64.argtypes = [C.c_uint32]
            L.o_mrg32k3a_to_f64.restype = C.c_double
            L.o_u32_to_f32.argtypes = [C.c_uint32]
            L.o_u32_to_f32.restype = C.c_float
            L.o_u32_to_f64.argtypes = [C.c_uint32]
            L.o_u32_to_f64.restype = C.c_double
            _lib = L
    return _lib


def gen_id(gen) -> int:
    return gen if isinstance(gen, int) else GEN_ID[gen.lower()]


def exp_bytes(n: int, nbytes: int | None = None) -> bytes:
    """Non-negative integer -> little-endian byte string for the jump functions."""
    if n < 0:
        raise ValueError("negative jump")
    need = max(1, (n.bit_length() + 7) // 8)
    return n.to_bytes(nbytes or need, "little")


def state_bytes(gen) -> int:
    return lib().oracle_state_bytes(gen_id(gen))


class State:
    """One generator state of the oracle (a single stream)."""

    def __init__(self, gen, seed: int):
        self.gen = gen_id(gen)
        self._buf = C.create_string_buffer(lib().oracle_internal_bytes(self.gen))
        if lib().oracle_seed(self.gen, seed, self._buf) != 0:
            raise ValueError(f"invalid seed {seed} for {GENS[self.gen]}")

    def jump(self, n: int) -> "State":
        e = exp_bytes(n)
        lib().oracle_jump(self.gen, self._buf, e, len(e))
        return self

    def fill(self, count: int, dtype: str = "u32") -> np.ndarray:
        code, npdt = DTYPES[dtype]
        out = np.empty(count, dtype=npdt)
        rc = lib().oracle_fill(self.gen, self._buf, count, code, out.ctypes.data, 1)
        assert rc == 0
        return out

    def export(self) -> bytes:
        out = C.create_string_buffer(lib().oracle_state_bytes(self.gen))
        lib().oracle_export(self.gen, self._buf, out)
        return out.raw

    def load(self, canon: bytes) -> "State":
        assert len(canon) == lib().oracle_state_bytes(self.gen)
        lib().oracle_import(self.gen, self._buf, canon)
        return self

    def copy(self) -> "State":
        other = object.__new__(State)
        other.gen = self.gen
        other._buf = C.create_string_buffer(self._buf.raw, len(self._buf))
        return other


def streams(gen, seed: int, s_first: int, s_count: int, block_len: int, n_per_stream: int,
            dtype: str = "u32", threads: int = 1, pre_jump: int = 0):
    """Block-split streams [s_first, s_first+s_count).

    Returns ``(out, states)``: ``out[i, j]`` = output number ``pre_jump + i`` of stream
    ``s_first + j`` (the canonical layout ``out[i*n_streams + s]`` restricted to these columns)
    and ``states[j]`` = canonical state bytes after the fill.  ``threads`` only splits the stream
    range over host threads (ctypes releases the GIL); the arithmetic stays scalar.
    """
    g = gen_id(gen)
    code, npdt = DTYPES[dtype]
    sb = lib().oracle_state_bytes(g)
    out = np.empty((n_per_stream, s_count), dtype=npdt)
    states = np.empty((s_count, sb), dtype=np.uint8)
    top = (s_first + max(s_count, 1) - 1) * block_len + pre_jump
    nb = max(1, (top.bit_length() + 7) // 8)

    def work(lo: int, hi: int):
        if hi <= lo:
            return 0
        e = b"".join(exp_bytes((s_first + j) * block_len + pre_jump, nb) for j in range(lo, hi))
        return lib().oracle_streams(g, seed, hi - lo, e, nb, n_per_stream, code,
                                    out.ctypes.data, s_count, lo,
                                    states[lo:hi].ctypes.data)

    if g == GEN_ID["mt19937"]:
        mt19937_charpoly()          # build the cached polynomial before any thread needs it
    threads = max(1, min(threads, s_count))
    if threads == 1:
        rcs = [work(0, s_count)]
    else:
        cuts = [s_count * t // threads for t in range(threads + 1)]
        with ThreadPoolExecutor(threads) as ex:
            rcs = list(ex.map(lambda ab: work(*ab), zip(cuts[:-1], cuts[1:])))
    if any(rcs):
        raise ValueError(f"oracle_streams failed: {rcs}")
    return out, states


def mt19937_charpoly():
    phi = np.zeros(312, dtype=np.uint64)
    deg = lib().o_mt19937_charpoly(phi.ctypes.data)
    return deg, phi


def mt19937_jump_poly(n: int) -> np.ndarray:
    g = np.zeros(312, dtype=np.uint64)
    e = exp_bytes(n)
    lib().o_mt19937_jump_poly(e, len(e), g.ctypes.data)
    return g


def gm_orbit(gen, seed: int, n: int):
    a, b = C.c_uint64(), C.c_uint64()
    e = exp_bytes(n)
    lib().o_gm_orbit(gen_id(gen), seed, e, len(e), C.byref(a), C.byref(b))
    return a.value, b.value
