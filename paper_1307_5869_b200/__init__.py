"""paper_1307_5869_b200 -- B200-native bulk multi-stream uniform RNG (PRAND, arXiv 1307.5869).

Thin ``ctypes`` binding of ``libprand.so`` (C ABI in ``include/prand.h``).  It marshals arguments
only: every step of the hot path (jump-ahead, recurrences, conversion, stores) runs in the library's
CUDA kernels.  The functions carry the C names; ``Generator`` is a small convenience wrapper that
takes torch tensors for device memory and CUDA streams.  There is no CPU fallback: if the library is
missing the import of any compute entry point raises.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libprand.so")

GENS = ["lfsr113", "mrg32k3a", "mt19937", "gm19", "gm29", "gm31", "gm55", "gm61",
        "gq58.1", "gq58.3", "gq58.4"]
GEN_ID = {name: i for i, name in enumerate(GENS)}
DTYPE_ID = {"u32": 0, "f32": 1, "f64": 2}

# include/prand.h: int prand_xxx(...) signatures
_SIGS = {
    "prand_init": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_uint64, C.c_uint64, C.c_uint64,
                             C.c_uint, C.c_void_p]),
    "prand_init_shard": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_uint64, C.c_uint64, C.c_uint64,
                                   C.c_uint64, C.c_uint, C.c_void_p]),
    "prand_jump": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint, C.c_void_p]),
    "prand_generate_u32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_f32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_f64": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_u32_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_f32_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_f64_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_state_bytes": (C.c_size_t, [C.c_void_p]),
    "prand_get_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "prand_set_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "prand_n_streams": (C.c_uint64, [C.c_void_p]),
    "prand_gen_of": (C.c_int, [C.c_void_p]),
    "prand_generate_seq_u32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_seq_f32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_seq_f64": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_lfsr113_seq_noalloc_u32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_state_device_ptr": (C.c_void_p, [C.c_void_p]),
    "prand_state_n_streams": (C.c_uint64, [C.c_void_p]),
    "prand_device_api_fill_u32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_device_api_fill_f32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_device_api_fill_f64": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_device_ops": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint, C.c_uint, C.POINTER(C.c_void_p), C.c_void_p]),
    "prand_device_api_init_fill_u32": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_device_api_init_fill_f32": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_device_api_init_fill_f64": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p]),
    "prand_generate_strided_u32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint, C.c_void_p]),
    "prand_generate_strided_f32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint, C.c_void_p]),
    "prand_generate_strided_f64": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint, C.c_void_p]),
    "prand_free": (C.c_int, [C.c_void_p]),
    "prand_fill_u32": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p]),
    "prand_probe_empty": (C.c_int, [C.c_void_p]),
    "prand_probe_memset": (C.c_int, [C.c_void_p, C.c_int, C.c_size_t, C.c_void_p]),
    "prand_probe_pipe_count": (C.c_int, []),
    "prand_probe_pipe_name": (C.c_char_p, [C.c_int]),
    "prand_probe_pipe": (C.c_int, [C.c_int, C.c_uint64, C.POINTER(C.c_uint64), C.c_void_p]),
    "prand_debug_set": (C.c_int, [C.c_char_p, C.c_char_p]),
    "prand_trim": (C.c_int, []),
    "prand_launch_count": (C.c_uint64, []),
    "prand_uploaded_bytes": (C.c_uint64, []),
    "prand_last_kernel": (C.c_char_p, [C.c_void_p]),
    "prand_strerror": (C.c_char_p, [C.c_int]),
    "prand_last_cuda_error": (C.c_int, []),
    "prand_version": (C.c_char_p, []),
    # include/prand_host.h
    "prand_host_skip_op_bytes": (C.c_size_t, [C.c_int]),
    "prand_host_skip_op": (C.c_int, [C.c_int, C.c_uint64, C.c_uint, C.c_void_p, C.c_size_t]),
    "prand_host_state_bytes": (C.c_size_t, [C.c_int]),
    "prand_host_seed_state": (C.c_int, [C.c_int, C.c_uint64, C.c_void_p, C.c_size_t]),
    "prand_host_mt19937_phi": (C.c_int, [C.c_void_p]),
    "prand_host_mt19937_phi_selfcheck": (C.c_int, []),
    "prand_host_mt19937_mulmod": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "prand_host_mt19937_table": (C.c_int, [C.c_uint64, C.c_uint, C.c_void_p]),
    "prand_host_gm_kq": (C.c_int, [C.c_int, C.c_uint64, C.c_uint, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]),
    "prand_host_plan_sections": (C.c_int, [C.c_int, C.c_uint64, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]),
    "prand_host_plan_sections_sm": (C.c_int, [C.c_int, C.c_uint64, C.c_int, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]),
    "prand_host_plan": (C.c_int, [C.c_int, C.c_uint64, C.c_uint64, C.c_int, C.c_int,
                                  C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]),
}
EXPORTS = sorted(_SIGS)

_lib = None


class PrandError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = lib().prand_strerror(code).decode()
        if code == -5:
            msg += f" (cudaError {lib().prand_last_cuda_error()})"
        super().__init__(f"{where}: {msg} [{code}]")


def lib() -> C.CDLL:
    """Load libprand.so (built in-tree by ``python -m paper_1307_5869_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1307_5869_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGS.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def gen_id(gen) -> int:
    return gen if isinstance(gen, int) else GEN_ID[gen.lower()]


def split_dist(n: int) -> tuple[int, int]:
    """Non-negative integer -> (mant, log2) with n = mant * 2^log2 and mant < 2^64."""
    if n < 0:
        raise ValueError("negative distance")
    if n == 0:
        return 0, 0
    log2 = (n & -n).bit_length() - 1
    mant = n >> log2
    if mant >> 64:
        raise ValueError("distance is not of the form mant * 2^log2 with mant < 2^64")
    return mant, log2


def _check(code: int, where: str) -> None:
    if code != 0:
        raise PrandError(code, where)


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


# ---- functions with the C names (argument marshalling only) --------------------------------------
def prand_init(gen, seed: int, n_streams: int, block_len: int, stream=None, first_stream: int = 0) -> int:
    """-> opaque state handle (int).  block_len is a Python int of the form mant * 2^log2."""
    mant, log2 = split_dist(block_len)
    h = C.c_void_p()
    _check(lib().prand_init_shard(C.byref(h), gen_id(gen), seed, first_stream, n_streams, mant, log2,
                                  _stream_ptr(stream)), "prand_init")
    return h.value


def prand_jump(state: int, steps: int, stream=None) -> None:
    mant, log2 = split_dist(steps)
    _check(lib().prand_jump(state, mant, log2, _stream_ptr(stream)), "prand_jump")


def _generate(name: str, state: int, out_ptr: int, n_per_stream: int, stream) -> None:
    _check(getattr(lib(), name)(state, out_ptr, n_per_stream, _stream_ptr(stream)), name)


def prand_generate_u32(state: int, out_ptr: int, n_per_stream: int, stream=None) -> None:
    _generate("prand_generate_u32", state, out_ptr, n_per_stream, stream)


def prand_generate_f32(state: int, out_ptr: int, n_per_stream: int, stream=None) -> None:
    _generate("prand_generate_f32", state, out_ptr, n_per_stream, stream)


def prand_generate_f64(state: int, out_ptr: int, n_per_stream: int, stream=None) -> None:
    _generate("prand_generate_f64", state, out_ptr, n_per_stream, stream)


def prand_generate_u32_host(state: int, host_ptr: int, n_per_stream: int, stream=None) -> None:
    _generate("prand_generate_u32_host", state, host_ptr, n_per_stream, stream)


def prand_generate_f32_host(state: int, host_ptr: int, n_per_stream: int, stream=None) -> None:
    _generate("prand_generate_f32_host", state, host_ptr, n_per_stream, stream)


def prand_generate_f64_host(state: int, host_ptr: int, n_per_stream: int, stream=None) -> None:
    _generate("prand_generate_f64_host", state, host_ptr, n_per_stream, stream)


def prand_get_state(state: int) -> bytes:
    n = lib().prand_state_bytes(state)
    buf = C.create_string_buffer(n)
    _check(lib().prand_get_state(state, buf, n), "prand_get_state")
    return buf.raw


def prand_set_state(state: int, canon: bytes) -> None:
    _check(lib().prand_set_state(state, canon, len(canon)), "prand_set_state")


def prand_lfsr113_seq_noalloc_u32(d_state_ptr: int, out_ptr: int, length: int, stream=None) -> None:
    """Single-sequence LFSR113 fill that allocates no device memory (include/prand.h): for callers that may not touch
    the CUDA allocator where they need the numbers.  ``d_state_ptr``: 4 u32 of the caller's device memory (canonical
    state, advanced in place); ``out_ptr``: ``length`` u32, 16-byte aligned; ``length`` <= NOALLOC_MAX_LENGTH."""
    _check(lib().prand_lfsr113_seq_noalloc_u32(d_state_ptr, out_ptr, length, _stream_ptr(stream)),
           "prand_lfsr113_seq_noalloc_u32")


NOALLOC_MAX_LENGTH = 1 << 31     # PRAND_NOALLOC_MAX_LENGTH of include/prand.h


def prand_free(state: int) -> None:
    _check(lib().prand_free(state), "prand_free")


def prand_fill_u32(out_ptr: int, n_words: int, value: int, stream=None) -> None:
    _check(lib().prand_fill_u32(out_ptr, n_words, value, _stream_ptr(stream)), "prand_fill_u32")


def prand_probe_empty(stream=None) -> None:
    _check(lib().prand_probe_empty(_stream_ptr(stream)), "prand_probe_empty")


def prand_probe_memset(ptr: int, value: int, nbytes: int, stream=None) -> None:
    _check(lib().prand_probe_memset(ptr, value, nbytes, _stream_ptr(stream)), "prand_probe_memset")


def prand_probe_pipe(op: int, iters: int, stream=None) -> int:
    """Launch instruction-rate probe `op`; -> thread-level operations the launch executes."""
    n = C.c_uint64()
    _check(lib().prand_probe_pipe(op, iters, C.byref(n), _stream_ptr(stream)), "prand_probe_pipe")
    return n.value


def prand_probe_pipe_names() -> list[str]:
    return [lib().prand_probe_pipe_name(i).decode() for i in range(lib().prand_probe_pipe_count())]


def prand_debug_set(name: str, value=None) -> None:
    """Set (value) or clear (None) one test / tuning hook of the library (include/prand.h)."""
    _check(lib().prand_debug_set(name.encode(), None if value is None else str(value).encode()), "prand_debug_set")


def prand_launch_count() -> int:
    return lib().prand_launch_count()


def prand_uploaded_bytes() -> int:
    return lib().prand_uploaded_bytes()


def prand_last_kernel(state: int) -> str:
    return lib().prand_last_kernel(state).decode()


# ---- host-only hooks (include/prand_host.h) -------------------------------------------------------
def prand_host_skip_op(gen, dist: int) -> bytes:
    g = gen_id(gen)
    mant, log2 = split_dist(dist)
    n = lib().prand_host_skip_op_bytes(g)
    buf = C.create_string_buffer(n)
    _check(lib().prand_host_skip_op(g, mant, log2, buf, n), "prand_host_skip_op")
    return buf.raw


def prand_host_seed_state(gen, seed: int) -> bytes:
    g = gen_id(gen)
    n = lib().prand_host_state_bytes(g)
    buf = C.create_string_buffer(n)
    _check(lib().prand_host_seed_state(g, seed, buf, n), "prand_host_seed_state")
    return buf.raw


def prand_host_mt19937_phi() -> bytes:
    buf = C.create_string_buffer(624 * 4)
    _check(lib().prand_host_mt19937_phi(buf), "prand_host_mt19937_phi")
    return buf.raw


def prand_host_mt19937_table(dist: int):
    """The precomputed polynomial of x^dist as bytes, or None if dist is not tabulated."""
    mant, log2 = split_dist(dist)
    buf = C.create_string_buffer(624 * 4)
    rc = lib().prand_host_mt19937_table(mant, log2, buf)
    return buf.raw if rc == 0 else None


def prand_host_mt19937_mulmod(a: bytes, b: bytes) -> bytes:
    buf = C.create_string_buffer(624 * 4)
    _check(lib().prand_host_mt19937_mulmod(a, b, buf), "prand_host_mt19937_mulmod")
    return buf.raw


def prand_host_plan(gen, n_streams: int, n_per_stream: int, dtype: str = "u32", sm_count: int = 148):
    cl, nc = C.c_uint64(), C.c_uint64()
    _check(lib().prand_host_plan(gen_id(gen), n_streams, n_per_stream, DTYPE_ID[dtype], sm_count,
                                 C.byref(cl), C.byref(nc)), "prand_host_plan")
    return cl.value, nc.value


# ---- convenience wrapper over torch tensors -------------------------------------------------------
class Generator:
    """``n_streams`` block-split streams of one generator on the current CUDA device.

    ``generate(n, dtype)`` returns a ``(n, n_streams)`` tensor whose element ``[i, s]`` is output
    number ``i`` (from the stream's current position) of stream ``s`` -- the canonical layout
    ``out[i * n_streams + s]`` of include/prand.h.
    """

    def __init__(self, gen, seed: int, n_streams: int, block_len: int, first_stream: int = 0, stream=None):
        self.gen = gen_id(gen)
        self.n_streams = n_streams
        self._h = prand_init(self.gen, seed, n_streams, block_len, stream, first_stream)

    def jump(self, steps: int, stream=None) -> None:
        prand_jump(self._h, steps, stream)

    def generate(self, n_per_stream: int, dtype: str = "u32", out=None, stream=None):
        import torch
        tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[dtype]
        if out is None:
            out = torch.empty((n_per_stream, self.n_streams), dtype=tdt, device="cuda")
        else:
            assert out.is_cuda and out.is_contiguous() and out.dtype == tdt
            assert out.numel() == n_per_stream * self.n_streams
        _generate("prand_generate_" + dtype, self._h, out.data_ptr(), n_per_stream, stream)
        return out

    def device_api_fill(self, n_per_stream: int, dtype: str = "u32", stream=None):
        """The library's example kernel written against include/prand_device.cuh (one thread per stream)."""
        import torch
        tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[dtype]
        out = torch.empty((n_per_stream, self.n_streams), dtype=tdt, device="cuda")
        _generate("prand_device_api_fill_" + dtype, self._h, out.data_ptr(), n_per_stream, stream)
        return out

    def device_api_init_fill(self, n_streams: int, block_len: int, n_per_stream: int, dtype: str = "u32", stream=None):
        """Streams initialised on the device by skip-ahead from this (one-stream) state: the library's example
        kernel for prand_device_ops + prand_dev::Gen<GEN>::skipahead."""
        import torch
        tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[dtype]
        out = torch.empty((n_per_stream, n_streams), dtype=tdt, device="cuda")
        mant, log2 = split_dist(block_len)
        _check(getattr(lib(), "prand_device_api_init_fill_" + dtype)(self._h, mant, log2, n_streams, out.data_ptr(),
                                                                     n_per_stream, _stream_ptr(stream)),
               "prand_device_api_init_fill")
        return out

    def generate_strided(self, n_per_stream: int, stride: int, dtype: str = "u32", stream=None):
        """Row i = every stream's output at its position + i * stride (the skip-per-step generator)."""
        import torch
        tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[dtype]
        out = torch.empty((n_per_stream, self.n_streams), dtype=tdt, device="cuda")
        mant, log2 = split_dist(stride)
        _check(getattr(lib(), "prand_generate_strided_" + dtype)(self._h, out.data_ptr(), n_per_stream, mant, log2,
                                                                 _stream_ptr(stream)), "prand_generate_strided")
        return out

    def generate_seq(self, length: int, dtype: str = "u32", out=None, stream=None):
        """PRAND's single-sequence fill (n_streams must be 1): the next ``length`` numbers, in order."""
        import torch
        tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[dtype]
        if out is None:
            out = torch.empty(length, dtype=tdt, device="cuda")
        else:
            assert out.is_cuda and out.is_contiguous() and out.dtype == tdt and out.numel() == length
        _generate("prand_generate_seq_" + dtype, self._h, out.data_ptr(), length, stream)
        return out

    def generate_host(self, n_per_stream: int, dtype: str = "u32", out=None, stream=None):
        """As ``generate`` but into HOST memory (pinned by default); returns after the data arrived."""
        import torch
        tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[dtype]
        if out is None:
            out = torch.empty((n_per_stream, self.n_streams), dtype=tdt, pin_memory=True)
        else:
            assert (not out.is_cuda) and out.is_contiguous() and out.dtype == tdt
        _generate("prand_generate_" + dtype + "_host", self._h, out.data_ptr(), n_per_stream, stream)
        return out

    def state(self) -> bytes:
        return prand_get_state(self._h)

    def set_state(self, canon: bytes) -> None:
        prand_set_state(self._h, canon)

    @property
    def last_kernel(self) -> str:
        return prand_last_kernel(self._h)

    def close(self) -> None:
        if self._h:
            prand_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
