"""GPU test of prand_lfsr113_seq_noalloc_u32, the entry point for callers that may not allocate device memory.

Some users of the library need random numbers at a point where the CUDA allocator is off limits: inside a
latency-critical loop that lives in one arena reserved at start-up, under a framework whose caching allocator owns
the device, in a plug-in that may only use buffers its host application passes in.  prand_init and
prand_generate_seq_* take device memory from the library's pool, so those users get one call that takes none: the
table of section start states and the jump operators sit in a fixed __device__ array inside libprand.so, the caller
passes the 16-byte generator state and the output array (include/prand.h).

What is checked: the numbers and the advanced state are bit for bit those of the existing path
(prand_init + prand_generate_seq_u32, itself compared with the oracle in test_gpu_parity.py), on two calls in a row
(the second call finds the first call's leftovers in the shared array and continues the sequence), for a length that
spans many sections with a ragged last one and for lengths shorter than one section; requests beyond the stated
capacity are refused.  The file sorts last on purpose (pytest -x stops at the first failure; nothing should hide
behind this one) and passes alone in a fresh process as well as after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1307_5869_b200 as P  # noqa: E402

SEED = 987654321


def need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def existing_path(pre_jump, lengths):
    """The numbers of prand_generate_seq_u32 on a one-stream state, call by call, and the canonical state after them."""
    g = P.Generator("lfsr113", SEED, 1, 0)
    if pre_jump:
        g.jump(pre_jump)
    start = g.state()
    outs = [g.generate_seq(n, "u32").cpu().numpy().view(np.uint32) for n in lengths]
    end = g.state()
    g.close()
    return start, outs, end


def no_alloc_path(start: bytes, lengths):
    """The same calls through the entry point that allocates nothing (the tensors here are the CALLER's memory)."""
    d_state = torch.from_numpy(np.frombuffer(start, dtype=np.int32).copy()).cuda()
    outs = []
    for n in lengths:
        out = torch.full((max(n, 1) + 8,), -1, dtype=torch.int32, device="cuda")      # 8 guard words behind the array
        P.prand_lfsr113_seq_noalloc_u32(d_state.data_ptr(), out.data_ptr(), n)
        torch.cuda.synchronize()
        host = out.cpu().numpy().view(np.uint32)
        assert (host[n:] == 0xFFFFFFFF).all(), "wrote past the end of the output array"
        outs.append(host[:n].copy())
    return outs, d_state.cpu().numpy().tobytes()


@pytest.mark.parametrize("lengths", [
    [3_000_017, 1_234_567],          # thousands of sections, ragged last section; second call continues the first
    [7, 1000, 33],                   # shorter than one section
    [70_000, 5],                     # a large call leaves a full table behind, the small one must not read it
])
def test_no_alloc_fill_equals_the_existing_path_on_two_calls_in_a_row(lengths):
    need_gpu()
    start, want, want_state = existing_path(12345, lengths)
    got, got_state = no_alloc_path(start, lengths)
    for i, (g, w) in enumerate(zip(got, want)):
        assert g.shape == w.shape
        assert np.array_equal(g, w), f"call {i} (length {lengths[i]}): {np.count_nonzero(g != w)} numbers differ"
    assert got_state == want_state


def test_no_alloc_fill_refuses_what_does_not_fit():
    need_gpu()
    L = P.lib()
    d_state = torch.from_numpy(np.frombuffer(P.Generator("lfsr113", SEED, 1, 0).state(), dtype=np.int32).copy()).cuda()
    before = d_state.cpu().numpy().tobytes()
    buf = torch.empty(64, dtype=torch.int32, device="cuda")
    too_long = P.NOALLOC_MAX_LENGTH + 1
    rc = L.prand_lfsr113_seq_noalloc_u32(d_state.data_ptr(), buf.data_ptr(), too_long, None)
    assert rc == -9 and b"capacity" in L.prand_strerror(rc)
    assert L.prand_lfsr113_seq_noalloc_u32(None, buf.data_ptr(), 16, None) == -2
    assert L.prand_lfsr113_seq_noalloc_u32(d_state.data_ptr(), None, 16, None) == -2
    assert L.prand_lfsr113_seq_noalloc_u32(d_state.data_ptr(), buf.data_ptr() + 4, 16, None) == -2    # not 16-byte aligned
    assert L.prand_lfsr113_seq_noalloc_u32(d_state.data_ptr(), None, 0, None) == 0                     # nothing to do
    torch.cuda.synchronize()
    assert d_state.cpu().numpy().tobytes() == before
